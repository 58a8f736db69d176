"""CPU-side checks of the C-ABI boundary: the shared library loads, exports every symbol
that include/pwa.h declares, refuses to run without a CUDA device (no CPU fallback), and its
host-only entry point (step A7) agrees with the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1108_5882_b200 import build
    build.build()
    from paper_1108_5882_b200 import binding as b
    return b


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "pwa.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pwa_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(binding):
    names = _declared_symbols()
    assert "pwa_create" in names and "pwa_nll_grad_batch" in names and len(names) >= 20
    lib = C.CDLL(binding.LIB_PATH)
    for name in names:
        assert hasattr(lib, name), f"{name} declared in pwa.h but not exported by libpwa.so"
    # and the binding wraps every one of them under the same name
    for name in names:
        assert name in binding.SYMBOLS
        assert hasattr(binding, name) or name in ("pwa_last_error", "pwa_status_string")


def test_no_torch_types_in_header():
    text = open(os.path.join(ROOT, "include", "pwa.h")).read()
    assert "torch" not in text.replace("torch.cuda.current_stream", "") and "at::" not in text


def test_create_fails_loudly_without_gpu(binding):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        pytest.skip("CUDA device present")
    with pytest.raises(binding.PwaError) as ei:
        binding.pwa_create(4, "f64")
    assert ei.value.status == binding.PWA_ERR_CUDA


def test_status_strings(binding):
    assert binding._status_name(binding.PWA_OK) == "PWA_OK"
    assert binding._status_name(binding.PWA_WARN_NONFINITE) == "PWA_WARN_NONFINITE"


def test_assemble_host_matches_oracle(binding, oracle):
    rng = np.random.default_rng(5)
    n = 7
    B = rng.normal(size=(500, n, 2)) * 0.3
    M = oracle.norm_matrix(B, 600)
    V, T = rng.normal(size=(n, 2)), rng.normal(size=(n, 2)) * 100
    L = -1234.5
    nll, g, parts = binding.pwa_assemble_host(L, T, M, V)
    nll_o, g_o, parts_o = oracle.assemble(L, T, M, V)
    assert nll == pytest.approx(nll_o, rel=1e-14)
    assert np.allclose(g, g_o, rtol=1e-13, atol=1e-13 * np.abs(g_o).max())
    assert np.allclose(parts, parts_o, rtol=1e-14)


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1108_5882_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp", ".c")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "pwa_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1108_5882_b200", text, flags=re.M), f
            assert "#include \"../paper" not in text and "csrc/" not in text.replace("paper_1108_5882_b200/csrc/,", ""), f


def test_eq2_and_polar_host_twins_match_oracle(binding):
    """NEXT-4: the host-only eq. 2 assembly and the polar chain rule against the oracle (no GPU)."""
    from oracle import oracle
    rng = np.random.default_rng(42)
    n, N = 6, 250
    A = rng.normal(size=(N, n, 2)) * 0.4
    B = rng.normal(size=(400, n, 2)) * 0.4
    V = rng.normal(size=(n, 2))
    M = oracle.norm_matrix(B, 450)
    L, T, _ = oracle.data_term(A, V)
    nll_o, g_o, parts_o = oracle.assemble_eq2(N, L, T, M, V)
    nll, g, parts = binding.pwa_assemble_host_eq2(N, L, T, M, V)
    assert nll == pytest.approx(nll_o, rel=1e-13) and np.allclose(parts, parts_o, rtol=1e-13)
    assert np.abs(g - g_o).max() <= 1e-12 * np.abs(g_o).max()
    gp = binding.pwa_grad_to_polar(V, g)
    assert np.abs(gp - oracle.grad_polar(V, g)).max() <= 1e-13 * np.abs(gp).max()
    r_phi = np.stack([np.hypot(V[:, 0], V[:, 1]), np.arctan2(V[:, 1], V[:, 0])], axis=-1)
    assert np.allclose(binding.pwa_polar_to_cartesian(r_phi), V, rtol=1e-14, atol=1e-15)


def test_fix_phase_host_matches_oracle(binding):
    """NEXT-4: the fixed-phase gauge (pwa_fix_phase_host, plain complex multiplication) against the oracle (angle
    arithmetic), including the gradient, a reference wave that is already real, V_ref = 0 and the argument checks."""
    from oracle import oracle
    rng = np.random.default_rng(43)
    n = 7
    for ref in (0, 4, n - 1):
        V, g = rng.normal(size=(n, 2)), rng.normal(size=(n, 2)) * 50.0
        V2, g2 = binding.pwa_fix_phase_host(V, g, ref)
        Vo, go = oracle.fix_phase(V, g, ref)
        assert np.abs(V2 - Vo).max() <= 1e-14 * np.abs(V).max() and np.abs(g2 - go).max() <= 1e-13 * np.abs(g).max()
        assert V2[ref, 1] == 0.0 and V2[ref, 0] > 0.0 and g2[ref, 1] == 0.0
        V3, none = binding.pwa_fix_phase_host(V2, None, ref)            # already in the gauge: unchanged to rounding
        assert none is None and np.abs(V3 - V2).max() <= 1e-15 * np.abs(V).max()
    V = rng.normal(size=(n, 2))
    V[2] = 0.0
    V2, g2 = binding.pwa_fix_phase_host(V, np.ones((n, 2)), 2)          # V_ref = 0: nothing to turn
    assert np.array_equal(V2, V) and g2[2, 1] == 0.0 and g2.sum() == 2 * n - 1
    for bad in (-1, n):
        with pytest.raises(binding.PwaError):
            binding.pwa_fix_phase_host(V, None, bad)
