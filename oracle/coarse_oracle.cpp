// coarse_oracle.cpp — CPU ORACLE for the coarse-grid Dirac operator apply.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
// shares no code with the CUDA path (paper_2212_12559_b200/csrc) and neither includes
// the other.
//
// What it computes (the plain definition, evaluated in fp64; nothing is blocked, fused
// or reordered beyond the definition):
//
//   O1 (non-dagger)  out(x) = X(x).in(x) + sum_{mu=0..3} [ Y_{+mu}(x).in(x+mu^) + Y_{-mu}(x).in(x-mu^) ]
//        BASELINE.json north_star; the paper names the operator ("coarse stencil
//        operator", §3.1) and its storage ("nine 48^2 matrices per
//        super-site: eight for the hopping terms and one for the [local] term",
//        PAPER.md:L101 §3.1) but never prints the formula (reading R1).
//   O2 (dagger)      out(x) = X(x)^H.in(x) + sum_mu [ Y_{+mu}(x-mu^)^H.in(x-mu^) + Y_{-mu}(x+mu^)^H.in(x+mu^) ]
//        the true adjoint of O1 for ARBITRARY links (needed because the setup solver
//        is CGNE, Table 1; reading R2).  Derivation:
//        A[x,x+mu^] = Y_{+mu}(x)  =>  A^H[y,y-mu^] = Y_{+mu}(y-mu^)^H, and
//        A[x,x-mu^] = Y_{-mu}(x)  =>  A^H[y,y+mu^] = Y_{-mu}(y+mu^)^H.
//   O4 (block)       nrhs independent single applies, one per right-hand side r
//        (multi-RHS is future work in the paper, §4.2; layout from
//        BASELINE.json config 5: site-major, RHS innermost).
//   O3 (int16 links) "the coarse links are stored in 16-bit fixed point format"
//        (PAPER.md:L99): entry = scale[s][m] * (q_re + i q_im), dequantised in double
//        ((double)q*(double)scale is exact) before the same loops run.
//   O5 (quantiser)   per matrix scale = max|component|/32767 (BASELINE.json config 4;
//        DESIGN.md readings R7, R8), q = clamp(rint(component/scale)) in fp32.
//
//   O7 (parts apply) the building block of the even/odd ("Schur-
//        preconditioned", Table 1) coarse operators.  With the site parity
//        pi(x) = (x0+x1+x2+x3) mod 2 and a parity set P (even, odd or all sites), for x in P
//            out(x) = alpha * Loc(x) + beta * Hop(x)
//            Loc(x) = X(x).u(x)  |  u(x) (identity)  |  0
//            Hop(x) = sum_mu [ Y_{+mu}(x).w(x+mu^) + Y_{-mu}(x).w(x-mu^) ]
//        and for dagger = 1 the same split of O2 (X^H u, and the adjoint hop).  Sites outside P
//        are not part of the result (returned as zero).  The Schur complement and its
//        block-preconditioned form are compositions of O7 written out in
//        oracle/__init__.py (schur_apply, schur_hat_apply) with numpy's dense solve as a step.
//
//   O8 (half-precision input vectors) PAPER.md:L97: "half precision" =
//        16-bit fixed point with a per-site fp32 norm.  Entry = norm[s][r] * (q_re + i q_im),
//        promoted in double before the same loops run; quantiser as O5 with one norm per (site, rhs).
//
// Layouts (identical to include/coarse_op.h because both take the caller's arrays):
//   site index s(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)); periodic wrap by modulo, so an
//   extent-2 direction adds both hops from the same neighbour and an extent-1 direction
//   adds both hops from the site itself (reading R13).
//   links[s][m][i][j], m = 0:X, 1+mu:Y_{+mu}, 5+mu:Y_{-mu}; out_i = sum_j M_ij in_j.
//   C64: float[2] (re,im).  I16: int16_t[2] (re,im) + scales[s][m] float.
//   vectors v[s][a][r] complex64 (float[2]), r innermost.  Output: complex128 (double[2]).
//
// Pins (-m "not gpu"): tests/test_oracle_pins.py - brute-force Galerkin P^H A P on tiny lattices
// (PAPER.md:L43), unit-shift cases, X-only vs a library einsum, dense assembly, adjoint identity,
// Gamma-Hermiticity, linearity, quantiser bounds; tests/test_oracle_evenodd_pins.py - O7
// against dense X / hopping blocks with parity masks, the dense Schur complement, the solution property;
// tests/test_oracle_hvec_pins.py - O8 against the complex64 apply on exactly representable data and the
// dense matrix; tests/test_oracle_cagcr_pins.py - the CA-GCR iterate (oracle/__init__.py) against scipy
// GMRES and the direct solve.  No function here or in oracle/__init__.py is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Lattice {
    int L[4];
    int64_t V;
};

inline void coords_of(const Lattice& lat, int64_t s, int x[4]) {
    x[0] = (int)(s % lat.L[0]); s /= lat.L[0];
    x[1] = (int)(s % lat.L[1]); s /= lat.L[1];
    x[2] = (int)(s % lat.L[2]); s /= lat.L[2];
    x[3] = (int)s;
}

inline int64_t index_of(const Lattice& lat, const int x[4]) {
    return x[0] + (int64_t)lat.L[0] * (x[1] + (int64_t)lat.L[1] * (x[2] + (int64_t)lat.L[2] * x[3]));
}

// site index of x + sign*mu^ with periodic wrap
inline int64_t neighbour(const Lattice& lat, int64_t s, int mu, int sign) {
    int x[4];
    coords_of(lat, s, x);
    x[mu] = ((x[mu] + sign) % lat.L[mu] + lat.L[mu]) % lat.L[mu];
    return index_of(lat, x);
}

// one link entry M(s,m)_ij as (re,im) in double, for either storage format
inline void link_entry(int prec, const void* links, const float* scales, int Nc,
                       int64_t s, int m, int i, int j, double& re, double& im) {
    const int64_t e = (((s * 9 + m) * Nc + i) * Nc + j) * 2;
    if (prec == 0) {
        const float* p = (const float*)links;
        re = (double)p[e];
        im = (double)p[e + 1];
    } else {
        const int16_t* p = (const int16_t*)links;
        const double sc = (double)scales[s * 9 + m];
        re = (double)p[e] * sc;
        im = (double)p[e + 1] * sc;
    }
}

// Half-precision input vectors (O8; "half precision ... 16-bit
// fixed point with a per-site fp32 norm"): when hv_q is set, the vector entry is
// (double)q[s][j][r] * (double)norm[s][r] instead of the float array handed to accumulate.
struct HalfVec {
    const int16_t* q = nullptr;     // int16 [V][Nc][nrhs][2]
    const float* norms = nullptr;   // float [V][nrhs]
};
thread_local HalfVec g_hv;

inline void vec_entry(const float* in, int Nc, int nrhs, int64_t sv, int j, int r, double& re, double& im) {
    const int64_t v = ((sv * Nc + j) * nrhs + r) * 2;
    if (g_hv.q) {
        const double n = (double)g_hv.norms[sv * nrhs + r];
        re = (double)g_hv.q[v] * n;
        im = (double)g_hv.q[v + 1] * n;
    } else {
        re = (double)in[v];
        im = (double)in[v + 1];
    }
}

// acc[i][r] += sum_j M(sm,m)_ij * in[sv][j][r]          (conj_transpose == 0)
// acc[i][r] += sum_j conj(M(sm,m)_ji) * in[sv][j][r]    (conj_transpose == 1)
void accumulate(int prec, const void* links, const float* scales, int Nc, int nrhs,
                int64_t sm, int m, int conj_transpose, const float* in, int64_t sv, double* acc) {
    for (int i = 0; i < Nc; ++i) {
        for (int j = 0; j < Nc; ++j) {
            double mre, mim;
            if (!conj_transpose) {
                link_entry(prec, links, scales, Nc, sm, m, i, j, mre, mim);
            } else {
                link_entry(prec, links, scales, Nc, sm, m, j, i, mre, mim);
                mim = -mim;
            }
            for (int r = 0; r < nrhs; ++r) {
                double vre, vim;
                vec_entry(in, Nc, nrhs, sv, j, r, vre, vim);
                acc[(i * nrhs + r) * 2 + 0] += mre * vre - mim * vim;
                acc[(i * nrhs + r) * 2 + 1] += mre * vim + mim * vre;
            }
        }
    }
}

// out_site[i][r] (complex128) for one output site s: definitions O1 / O2
void apply_site(const Lattice& lat, int Nc, int prec, const void* links, const float* scales,
                const float* in, int nrhs, int dagger, int64_t s, double* out_site) {
    std::memset(out_site, 0, sizeof(double) * 2 * Nc * nrhs);
    if (!dagger) {
        accumulate(prec, links, scales, Nc, nrhs, s, 0, 0, in, s, out_site);                 // X(x) in(x)
        for (int mu = 0; mu < 4; ++mu) {
            const int64_t fwd = neighbour(lat, s, mu, +1), bwd = neighbour(lat, s, mu, -1);
            accumulate(prec, links, scales, Nc, nrhs, s, 1 + mu, 0, in, fwd, out_site);      // Y_{+mu}(x) in(x+mu^)
            accumulate(prec, links, scales, Nc, nrhs, s, 5 + mu, 0, in, bwd, out_site);      // Y_{-mu}(x) in(x-mu^)
        }
    } else {
        accumulate(prec, links, scales, Nc, nrhs, s, 0, 1, in, s, out_site);                 // X(x)^H in(x)
        for (int mu = 0; mu < 4; ++mu) {
            const int64_t fwd = neighbour(lat, s, mu, +1), bwd = neighbour(lat, s, mu, -1);
            accumulate(prec, links, scales, Nc, nrhs, bwd, 1 + mu, 1, in, bwd, out_site);    // Y_{+mu}(x-mu^)^H in(x-mu^)
            accumulate(prec, links, scales, Nc, nrhs, fwd, 5 + mu, 1, in, fwd, out_site);    // Y_{-mu}(x+mu^)^H in(x+mu^)
        }
    }
}

// O7 for one output site: out_site = alpha*Loc + beta*Hop (see the header).
//   local: 0 none, 1 X (X^H for dagger), 2 identity.
void parts_site(const Lattice& lat, int Nc, int prec, const void* links, const float* scales,
                const float* u, const float* w, int nrhs, int dagger, int local, double alpha,
                double beta, int64_t s, double* out_site, double* tmp) {
    const int64_t n = (int64_t)2 * Nc * nrhs;
    std::memset(out_site, 0, sizeof(double) * n);
    // local term
    std::memset(tmp, 0, sizeof(double) * n);
    if (local == 1) {
        accumulate(prec, links, scales, Nc, nrhs, s, 0, dagger, u, s, tmp);
    } else if (local == 2) {
        for (int64_t e = 0; e < n; ++e) tmp[e] = (double)u[s * n + e];
    }
    for (int64_t e = 0; e < n; ++e) out_site[e] += alpha * tmp[e];
    // hopping term
    std::memset(tmp, 0, sizeof(double) * n);
    for (int mu = 0; mu < 4; ++mu) {
        const int64_t fwd = neighbour(lat, s, mu, +1), bwd = neighbour(lat, s, mu, -1);
        if (!dagger) {
            accumulate(prec, links, scales, Nc, nrhs, s, 1 + mu, 0, w, fwd, tmp);      // Y_{+mu}(x) w(x+mu^)
            accumulate(prec, links, scales, Nc, nrhs, s, 5 + mu, 0, w, bwd, tmp);      // Y_{-mu}(x) w(x-mu^)
        } else {
            accumulate(prec, links, scales, Nc, nrhs, bwd, 1 + mu, 1, w, bwd, tmp);    // Y_{+mu}(x-mu^)^H w(x-mu^)
            accumulate(prec, links, scales, Nc, nrhs, fwd, 5 + mu, 1, w, fwd, tmp);    // Y_{-mu}(x+mu^)^H w(x+mu^)
        }
    }
    for (int64_t e = 0; e < n; ++e) out_site[e] += beta * tmp[e];
}

inline int site_parity(const Lattice& lat, int64_t s) {
    int x[4];
    coords_of(lat, s, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
}

bool valid(const int dims[4], int Nc, int prec, int nrhs, int dagger) {
    if (!dims || Nc < 1 || nrhs < 1) return false;
    if (prec != 0 && prec != 1) return false;
    if (dagger != 0 && dagger != 1) return false;
    for (int mu = 0; mu < 4; ++mu) if (dims[mu] < 1) return false;
    return true;
}

}  // namespace

extern "C" {

// Threads an apply with nthreads <= 0 would use.
int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Full-lattice apply.  out is complex128 [V][Nc][nrhs].  Returns 0, or -1 on bad arguments.
// nthreads <= 0: all cores OpenMP reports.  The parallel loop is over output sites only.
int oracle_coarse_apply(const int dims[4], int Nc, int link_precision, const void* links,
                        const float* scales, const float* in, double* out, int nrhs, int dagger,
                        int nthreads) {
    if (!valid(dims, Nc, link_precision, nrhs, dagger) || !links || !in || !out) return -1;
    if (link_precision == 1 && !scales) return -1;
    Lattice lat{{dims[0], dims[1], dims[2], dims[3]}, (int64_t)dims[0] * dims[1] * dims[2] * dims[3]};
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (int64_t s = 0; s < lat.V; ++s)
        apply_site(lat, Nc, link_precision, links, scales, in, nrhs, dagger, s,
                   out + s * 2 * (int64_t)Nc * nrhs);
    return 0;
}

// The same definition evaluated only at the listed output sites:
// out is complex128 [nsites][Nc][nrhs], row k holding out(sites[k]).
int oracle_coarse_apply_sites(const int dims[4], int Nc, int link_precision, const void* links,
                              const float* scales, const float* in, double* out, int nrhs,
                              int dagger, const int64_t* sites, int64_t nsites, int nthreads) {
    if (!valid(dims, Nc, link_precision, nrhs, dagger) || !links || !in || !out || !sites) return -1;
    if (link_precision == 1 && !scales) return -1;
    Lattice lat{{dims[0], dims[1], dims[2], dims[3]}, (int64_t)dims[0] * dims[1] * dims[2] * dims[3]};
    for (int64_t k = 0; k < nsites; ++k) if (sites[k] < 0 || sites[k] >= lat.V) return -1;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (int64_t k = 0; k < nsites; ++k)
        apply_site(lat, Nc, link_precision, links, scales, in, nrhs, dagger, sites[k],
                   out + k * 2 * (int64_t)Nc * nrhs);
    return 0;
}

// O7: parts apply.  parity: 0 even sites, 1 odd sites, 2 all sites; local: 0 none, 1 X, 2 identity.
// u may be NULL when local == 0.  out is complex128 [V][Nc][nrhs]; sites outside the parity set are 0.
int oracle_coarse_apply_parts(const int dims[4], int Nc, int link_precision, const void* links,
                              const float* scales, const float* u, const float* w, double* out,
                              int nrhs, int dagger, int parity, int local, double alpha, double beta,
                              int nthreads) {
    if (!valid(dims, Nc, link_precision, nrhs, dagger) || !links || !w || !out) return -1;
    if (link_precision == 1 && !scales) return -1;
    if (parity < 0 || parity > 2 || local < 0 || local > 2) return -1;
    if (local != 0 && !u) return -1;
    Lattice lat{{dims[0], dims[1], dims[2], dims[3]}, (int64_t)dims[0] * dims[1] * dims[2] * dims[3]};
    const int64_t n = (int64_t)2 * Nc * nrhs;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel num_threads(nthreads)
#endif
    {
        double* tmp = new double[n];
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t s = 0; s < lat.V; ++s) {
            if (parity != 2 && site_parity(lat, s) != parity) {
                std::memset(out + s * n, 0, sizeof(double) * n);
                continue;
            }
            parts_site(lat, Nc, link_precision, links, scales, u, w, nrhs, dagger, local, alpha, beta, s,
                       out + s * n, tmp);
        }
        delete[] tmp;
    }
    return 0;
}

// O8: the full apply (O1/O2) on half-precision INPUT vectors: in(x)_jr = q[x][j][r] * norm[x][r].
// Output complex128 as always.
int oracle_coarse_apply_hvec(const int dims[4], int Nc, int link_precision, const void* links,
                             const float* scales, const int16_t* in_q, const float* in_norms, double* out,
                             int nrhs, int dagger, int nthreads) {
    if (!valid(dims, Nc, link_precision, nrhs, dagger) || !links || !in_q || !in_norms || !out) return -1;
    if (link_precision == 1 && !scales) return -1;
    Lattice lat{{dims[0], dims[1], dims[2], dims[3]}, (int64_t)dims[0] * dims[1] * dims[2] * dims[3]};
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel num_threads(nthreads)
#endif
    {
        g_hv.q = in_q;
        g_hv.norms = in_norms;
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t s = 0; s < lat.V; ++s)
            apply_site(lat, Nc, link_precision, links, scales, nullptr, nrhs, dagger, s,
                       out + s * 2 * (int64_t)Nc * nrhs);
        g_hv = HalfVec();
    }
    return 0;
}

// O8 evaluated only at the listed output sites (the same apply_site as every other entry point):
// out is complex128 [nsites][Nc][nrhs], row k holding out(sites[k]).
int oracle_coarse_apply_hvec_sites(const int dims[4], int Nc, int link_precision, const void* links,
                                   const float* scales, const int16_t* in_q, const float* in_norms, double* out,
                                   int nrhs, int dagger, const int64_t* sites, int64_t nsites, int nthreads) {
    if (!valid(dims, Nc, link_precision, nrhs, dagger) || !links || !in_q || !in_norms || !out || !sites) return -1;
    if (link_precision == 1 && !scales) return -1;
    Lattice lat{{dims[0], dims[1], dims[2], dims[3]}, (int64_t)dims[0] * dims[1] * dims[2] * dims[3]};
    for (int64_t k = 0; k < nsites; ++k) if (sites[k] < 0 || sites[k] >= lat.V) return -1;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel num_threads(nthreads)
#endif
    {
        g_hv.q = in_q;
        g_hv.norms = in_norms;
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int64_t k = 0; k < nsites; ++k)
            apply_site(lat, Nc, link_precision, links, scales, nullptr, nrhs, dagger, sites[k],
                       out + k * 2 * (int64_t)Nc * nrhs);
        g_hv = HalfVec();
    }
    return 0;
}

// O8 quantiser for vectors: one fp32 norm per (site, right-hand side),
//   amax = max over the 2*Nc real components of |component|, norm = amax / 32767.0f,
//   q = (int16) clamp(nearbyintf(component / norm), -32767, 32767); amax == 0 => norm = 0, q = 0.
// v: float [n_sites][Nc][nrhs][2]; q: int16 same shape; norms: float [n_sites][nrhs].
int oracle_quantize_vec_i16(const float* v, int64_t n_sites, int Nc, int nrhs, int16_t* q, float* norms) {
    if (!v || !q || !norms || n_sites < 0 || Nc < 1 || nrhs < 1) return -1;
    for (int64_t s = 0; s < n_sites; ++s)
        for (int r = 0; r < nrhs; ++r) {
            float amax = 0.0f;
            for (int a = 0; a < Nc; ++a)
                for (int c = 0; c < 2; ++c) amax = std::max(amax, std::fabs(v[((s * Nc + a) * nrhs + r) * 2 + c]));
            const float norm = amax == 0.0f ? 0.0f : amax / 32767.0f;
            norms[s * nrhs + r] = norm;
            for (int a = 0; a < Nc; ++a)
                for (int c = 0; c < 2; ++c) {
                    const int64_t e = ((s * Nc + a) * nrhs + r) * 2 + c;
                    if (amax == 0.0f) { q[e] = 0; continue; }
                    float t = nearbyintf(v[e] / norm);
                    t = std::min(32767.0f, std::max(-32767.0f, t));
                    q[e] = (int16_t)t;
                }
        }
    return 0;
}

// Site indices of the stencil of site s: nbr[0]=s, nbr[1+mu]=s(x+mu^), nbr[5+mu]=s(x-mu^).
int oracle_neighbours(const int dims[4], int64_t s, int64_t nbr[9]) {
    if (!dims || !nbr) return -1;
    for (int mu = 0; mu < 4; ++mu) if (dims[mu] < 1) return -1;
    Lattice lat{{dims[0], dims[1], dims[2], dims[3]}, (int64_t)dims[0] * dims[1] * dims[2] * dims[3]};
    if (s < 0 || s >= lat.V) return -1;
    nbr[0] = s;
    for (int mu = 0; mu < 4; ++mu) {
        nbr[1 + mu] = neighbour(lat, s, mu, +1);
        nbr[5 + mu] = neighbour(lat, s, mu, -1);
    }
    return 0;
}

// O5: int16 fixed-point quantiser, one fp32 scale per Nc x Nc matrix.
//   amax  = max over the 2*Nc^2 real components of |component|          (fp32)
//   scale = amax / 32767.0f                                              (one fp32 division)
//   q     = (int16) clamp(nearbyintf(component / scale), -32767, 32767)  (fp32, round-half-even)
//   amax == 0  =>  scale = 0 and every q = 0.   -32768 is never produced.
// links: float[n_matrices][Nc][Nc][2]; q: int16[n_matrices][Nc][Nc][2]; scales: float[n_matrices].
int oracle_quantize_i16(const float* links, int64_t n_matrices, int Nc, int16_t* q, float* scales) {
    if (!links || !q || !scales || n_matrices < 0 || Nc < 1) return -1;
    const int64_t per = (int64_t)2 * Nc * Nc;
    for (int64_t k = 0; k < n_matrices; ++k) {
        const float* src = links + k * per;
        int16_t* dst = q + k * per;
        float amax = 0.0f;
        for (int64_t e = 0; e < per; ++e) amax = std::max(amax, std::fabs(src[e]));
        if (amax == 0.0f) {
            scales[k] = 0.0f;
            for (int64_t e = 0; e < per; ++e) dst[e] = 0;
            continue;
        }
        const float scale = amax / 32767.0f;
        scales[k] = scale;
        for (int64_t e = 0; e < per; ++e) {
            float t = nearbyintf(src[e] / scale);     // default rounding mode: to nearest even
            t = std::min(32767.0f, std::max(-32767.0f, t));
            dst[e] = (int16_t)t;
        }
    }
    return 0;
}

// Dequantise to double: entry = (double)q * (double)scale (exact).  out: double[n_matrices][Nc][Nc][2].
int oracle_dequantize_i16(const int16_t* q, const float* scales, int64_t n_matrices, int Nc, double* out) {
    if (!q || !scales || !out || n_matrices < 0 || Nc < 1) return -1;
    const int64_t per = (int64_t)2 * Nc * Nc;
    for (int64_t k = 0; k < n_matrices; ++k)
        for (int64_t e = 0; e < per; ++e)
            out[k * per + e] = (double)q[k * per + e] * (double)scales[k];
    return 0;
}

}  // extern "C"
