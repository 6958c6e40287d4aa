"""CPU-side check that the built library is sm_100a-native: its SASS holds the tcgen05 / TMEM / TMA instructions the
kernels are written with (tcgen05.mma kind::tf32 -> UTCHMMA, kind::i8 -> UTCIMMA, tcgen05.ld / st -> LDTM / STTM,
cp.async.bulk(.tensor) -> UBLKCP / UTMALDG) and no legacy mma.sync (HMMA).  Needs cuobjdump, no GPU."""
import shutil
import subprocess

import pytest

from paper_2212_12559_b200 import build as cuda_build
from paper_2212_12559_b200 import sass_counts


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not installed")
def test_library_sass_is_blackwell_native():
    """Two of the library's translation units (disassembling all 27 takes minutes): the Nc = 128 tensor kernels and the
    Nc = 48 streaming kernels - BASELINE configs C5 and C2."""
    import os
    cuda_build.build_library()
    objs = [os.path.join(cuda_build.OBJ_DIR, n) for n in ("launch_tensor_nc128.o", "launch_stream_nc48.o")]
    if not all(os.path.exists(o) for o in objs):
        cuda_build.build_library(force=True)
    sass = "".join(subprocess.run(["cuobjdump", "-sass", o], capture_output=True, text=True, check=True).stdout for o in objs)
    counts = {k: 0 for k in sass_counts.COLS}
    archs = set()
    for line in sass.splitlines():
        m = sass_counts.PAT.search(line)
        if m:
            counts[m.group(1)] += 1
        if "arch = sm_" in line:
            archs.add(line.split("arch = ")[1].strip())
    assert archs == {"sm_100a"}, archs
    for k in ("UTCHMMA", "UTCIMMA", "UTCBAR", "LDTM", "STTM", "UTMALDG", "UBLKCP", "SYNCS", "FFMA2"):
        assert counts[k] > 0, (k, counts)
    assert counts["HMMA"] == 0


def test_kernel_family_names():
    assert sass_counts.family("_ZN6coarse22coarse_apply_tensor_i8ILi128ELi16ELb0EEEv14CUtensorMap_stNS_14TensorI8ParamsE") == "coarse_apply_tensor_i8"
    assert sass_counts.family("_ZN6coarse20coarse_apply_stream2ILi64ELb1ELb0ELi4EEEvNS_12StreamParamsE") == "coarse_apply_stream2"
    assert sass_counts.family("_ZN6coarse17cagcr_gram_kernelENS_9CagcrVecsExiP7double2") == "cagcr_gram_kernel"
