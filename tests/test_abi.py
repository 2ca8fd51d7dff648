"""Host-side checks of the C-ABI library (no GPU needed): it builds, loads, exports every symbol that
include/ea.h declares, and fails loudly -- never falls back -- when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest

from paper_1411_5512_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ea.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ea_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_all_exported_and_bound(lib):
    names = declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), "libea_b200.so does not export %s" % n
        assert n in binding.SIGNATURES, "binding.py does not marshal %s" % n
    assert sorted(binding.SIGNATURES) == names


def test_library_links_no_python_or_torch():
    import subprocess
    out = subprocess.run(["ldd", binding.LIB_PATH], capture_output=True, text=True).stdout
    names = [line.split()[0] for line in out.splitlines() if line.strip()]
    assert names and not any("torch" in n or "python" in n or "c10" in n for n in names), names


def test_library_holds_sm100a_code():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_workspace_bytes_and_argument_validation(lib):
    assert lib.ea_workspace_bytes(3, 1, 0) == 0          # odd L
    assert lib.ea_workspace_bytes(0, 1, 0) == 0
    assert lib.ea_workspace_bytes(8, 3, 0) == 0          # n_replicas
    assert lib.ea_workspace_bytes(8, 1, -1) == 0
    assert lib.ea_workspace_bytes(2048, 1, 0) == 0       # L^3 >= 2^31
    n1 = lib.ea_workspace_bytes(128, 1, 2)
    n2 = lib.ea_workspace_bytes(128, 2, 2)
    N = 128 ** 3
    assert n1 >= N * 8 * (1 + 3 + 2 + 1) and n1 < N * 8 * 7 + (1 << 20)
    assert n1 - n2 == 3 * N * 4                          # 32-bit bond words in replica mode
    h = C.c_void_p()
    bad = [(7, 0.5, 0.8, 64), (8, 1.5, 0.8, 64), (8, 0.5, -1.0, 64), (8, 0.5, 0.8, 48), (8, 0.5, 0.8, 8),
           (8, float("nan"), 0.8, 64)]  # n_samples 48: not 2^m; 8 at L = 8: one plane per slab (needs an even number)
    for L, p, T, ns in bad:
        assert lib.ea_create(L, p, T, ns, 1, C.byref(h)) == binding.EA_ERR_INVALID
    assert lib.ea_strerror(binding.EA_ERR_STATE) == b"invalid state"
    assert b"sm_100a" in lib.ea_version()


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the GPU-less box")
    h = C.c_void_p()
    assert lib.ea_create(8, 0.5, 0.8, 64, 1, C.byref(h)) == binding.EA_ERR_CUDA
    with pytest.raises(binding.EAError):
        binding.Sim(8, 0.5, 0.8)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1411_5512_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "ea_oracle" not in src, f


def test_host_side_c4_curve_and_integral_estimator_match_the_oracle():
    """ea_c4_curve / ea_integral_estimator do no device work (double arithmetic on the host, Eq. 5-6 and the
    procedure of PAPER.md:116): compared here, without a GPU, with the oracle's fp64 restatement; 1e-12 relative."""
    import numpy as np
    import oracle
    from paper_1411_5512_b200 import binding
    rng = np.random.default_rng(11)
    R, N = 6, 4096
    n_bins = 3 * R * R + 1
    mult = np.zeros(n_bins, dtype=np.int64)
    for dz in range(-R, R + 1):
        for dy in range(-R, R + 1):
            for dx in range(-R, R + 1):
                mult[dx * dx + dy * dy + dz * dz] += 1
    r_all = np.sqrt(np.arange(n_bins))
    base = N * np.exp(-r_all / 1.7)
    S = np.rint((base[:, None] + rng.normal(0, 600.0, size=(n_bins, 32))) * mult[:, None]).astype(np.int64)
    for r_lim in (R, 3):
        got = binding.c4_curve(S, mult, N, r_lim)
        want = oracle.c4_curve(S, mult, N, r_lim)
        assert len(got[0]) == len(want[0]) > 3
        for a, b in zip(got, want):
            np.testing.assert_allclose(a, b, rtol=1e-12, atol=0)
    r, c, e = oracle.c4_curve(S, mult, N, R)
    for k in (0, 1, 2):
        got = binding.integral_estimator(r, c, e, k)
        want = oracle.integral_estimator(r, c, e, k)
        np.testing.assert_allclose(got, want, rtol=1e-12, atol=0)
    assert binding.integral_estimator(r, c, e, 1)[3] < R          # the noisy tail is cut off
    got = binding.integral_estimator(r, np.abs(c) + 1e-9, np.zeros_like(e), 1)    # nothing below 3 e: no cut-off
    assert got[3] == r[-1]


def test_workspace_bytes_ex_validates_the_mixed_coding_parameters():
    """No device needed: sizes and the validity rule of n_samples = M < 64 (DESIGN.md C-M)."""
    from paper_1411_5512_b200 import binding
    f = binding.lib().ea_workspace_bytes_ex
    base = binding.lib().ea_workspace_bytes(16, 2, 1)
    assert f(16, 64, 2, 1) == base > 0
    assert f(16, 32, 2, 1) >= base + (16 ** 3 // 2) * 4 * 8        # folded spins + 3 folded bond planes, K = 2
    assert f(16, 8, 2, 1) > base
    for L, M, n_rep in ((10, 32, 2), (16, 3, 2), (16, 1, 2), (8, 8, 2), (16, 128, 2), (16, 0, 1)):
        assert f(L, M, n_rep, 1) == 0
    assert f(128, 1, 1, 0) > 0                                     # one sample, 64 slabs of two planes


def test_resident_row_schedules_are_consistent_on_the_host():
    """The RESIDENT kernel's host-built row tables satisfy their invariants; no device needed."""
    from paper_1411_5512_b200 import binding
    assert binding.lib().ea_selftest_host() == binding.EA_OK


def test_pipe_microbenchmark_streams_hold_exactly_the_counted_instructions():
    """ea_selftest_pipes reports warp instructions per second; the count it divides by is 8 (ILP) x 16 (unroll) per
    loop trip.  Checked here, without a GPU, in the SASS of the library: each stream's loop body holds exactly 128
    instructions of its kind (LOP3 / IMAD.WIDE.U32 / POPC; the mixes hold 128 + 32 IMAD.WIDE and 128 + 128 IMAD) -- ptxas has not folded any."""
    import subprocess
    want = {0: {"LOP3": 128}, 1: {"IMAD.WIDE": 128}, 2: {"POPC": 128}, 3: {"LOP3": 128, "IMAD.WIDE": 32}, 4: {"LOP3": 128, "IMAD": 128}}
    for kind, ops in want.items():
        name = "_ZN2ea13k_pipe_streamILi%dEEEvPjiPy" % kind
        out = subprocess.run(["cuobjdump", "-sass", "-fun", name, binding.LIB_PATH], capture_output=True, text=True).stdout
        lines = [m.groups() for m in re.finditer(r"/\*([0-9a-f]{4})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)([^;]*);", out)]
        assert lines, "kernel %s not found in the library" % name
        # the timed loop = from the target of the one backward branch to that branch
        back = [(int(a, 16), int(re.search(r"0x([0-9a-f]+)", rest).group(1), 16)) for a, op, rest in lines
                if op.startswith("BRA") and re.search(r"0x([0-9a-f]+)", rest) and int(re.search(r"0x([0-9a-f]+)", rest).group(1), 16) < int(a, 16)]
        assert len(back) == 1, back
        hi, lo = back[0]
        body = [op for a, op, _ in lines if lo <= int(a, 16) <= hi]
        for op, n in ops.items():
            assert sum(1 for o in body if o.startswith(op)) == n, (kind, op, sum(1 for o in body if o.startswith(op)))
