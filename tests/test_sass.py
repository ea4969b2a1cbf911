"""What the compiled library contains (no GPU needed): the hot kernel is sm_100a code that uses the hardware features
DESIGN.md section 6 names -- TMA box loads and bulk copies, mbarrier waits, packed FFMA2, vector reductions,
setmaxnreg, elect -- and neither of its two shapes spills registers (the consumers sit at their register budget:
a change that makes ptxas spill inside the frame loop costs several per cent, profiles/r2_fma_ceiling.md)."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _cuobjdump():
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not found")
    return exe


@pytest.fixture(scope="module")
def sass():
    import __graft_entry__
    __graft_entry__.build()
    from paper_2209_09848_b200 import binding
    out = subprocess.run([_cuobjdump(), "-sass", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in out or "SM100a" in out.upper() or "sm_100" in out
    # function name -> its SASS text
    parts = re.split(r"\n\s*Function : ", out)
    return {p.split("\n", 1)[0].strip(): p for p in parts[1:]}


def _kernels(sass, needle):
    return {k: v for k, v in sass.items() if needle in k}


def test_library_is_sm100a_only(sass):
    exe = _cuobjdump()
    from paper_2209_09848_b200 import binding
    lst = subprocess.run([exe, "-lelf", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", lst))
    assert archs == {"100a"}, archs


def test_search_kernel_uses_tma_mbarriers_ffma2_and_vector_reductions(sass):
    ks = _kernels(sass, "k_search_sep")
    assert len(ks) == 2, list(ks)                       # the two kernel shapes
    for name, text in ks.items():
        for mnemonic in ("UTMALDG.3D", "UBLKCP", "SYNCS.PHASECHK.TRANS64.TRYWAIT", "SYNCS.ARRIVE", "FFMA2", "FADD2",
                         "REDG.E.ADD.F32x2", "USETMAXREG", "ELECT"):
            assert mnemonic in text, (name[:60], mnemonic)
        # the y-pass: 5 FFMA2 per position and slot (4 x 5 or 5 x 4 of them), once for full and once for partial
        # batches, + the 8 exact differences
        assert text.count("FFMA2") >= 2 * 100 + 8, (name[:60], text.count("FFMA2"))


def test_search_kernel_does_not_spill(sass):
    for name, text in _kernels(sass, "k_search_sep").items():
        assert not re.search(r"\b(STL|LDL)\b", text), name[:60]
