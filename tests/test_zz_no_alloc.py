"""pwa_data_term_static: the allocation-free entry point (static device scratch, no context) against the existing context
path (pwa_data_term_enqueue) on the same device buffers, two calls in a row, at the tolerance of the other GPU tests
(1e-12 fp64 storage / 1e-6 fp32 storage, norm-wise, reading C8), and against the oracle.  Collected last on purpose (the
suite runs with pytest -x).  Passes alone in a fresh process and after the other tests: nothing here depends on state
another test leaves, and the shared static array is cleared by every call as far as it must start at zero.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-6}


@pytest.fixture(scope="module")
def pwa():
    from paper_1108_5882_b200 import binding
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    return binding


def _case(seed, N, n, storage):
    rng = np.random.default_rng(seed)
    A = (rng.normal(size=(N, n, 2)) * 0.35).astype(np.float64 if storage == "f64" else np.float32)
    return A, rng.normal(size=(2, n, 2))


def _close(rec, ref, tol):
    """records {L_data, n_nonfinite, T}: |dL| <= tol |L_data|, the count equal, |dT|_max <= tol |T|_max"""
    assert abs(rec[0] - ref[0]) <= tol * abs(ref[0]), ("L_data", rec[0], ref[0])
    assert rec[1] == ref[1]
    assert np.abs(rec[2:] - ref[2:]).max() <= tol * np.abs(ref[2:]).max(), ("T", np.abs(rec[2:] - ref[2:]).max() / np.abs(ref[2:]).max())


@pytest.mark.parametrize("storage,n,N", [("f64", 5, 7001), ("f64", 16, 100_003), ("f32", 32, 50_001), ("f32", 64, 200_003),
                                         ("f64", 64, 131), ("f32", 1, 1)])
def test_static_entry_point_matches_context_path(pwa, oracle, storage, n, N):
    import torch
    A, Vs = _case(900 + n, N, n, storage)
    A_dev = torch.from_numpy(A).cuda()
    stream = torch.cuda.current_stream().cuda_stream
    ref_dev = torch.zeros(2 + 2 * n, dtype=torch.float64, device="cuda")
    refs = []
    ctx = pwa.pwa_create(n, storage, 0, stream)
    try:
        pwa.pwa_upload_events(ctx, pwa.PWA_DATA, A_dev, n_events=N, flags=pwa.PWA_BORROW)
        for V in Vs:
            pwa.pwa_data_term_enqueue(ctx, V, ref_dev)
            refs.append(ref_dev.cpu().numpy().copy())
    finally:
        pwa.pwa_destroy(ctx)
    # two calls in a row through the static entry point (the second finds the first one's partials in the array)
    out_a = torch.full((2 + 2 * n,), float("nan"), dtype=torch.float64, device="cuda")
    out_b = torch.full((2 + 2 * n,), float("nan"), dtype=torch.float64, device="cuda")
    pwa.pwa_data_term_static(A_dev, Vs[0], out_a, cuda_stream=stream)          # first call on this device: symbol look-up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    pwa.pwa_data_term_static(A_dev, Vs[0], out_a, cuda_stream=stream)
    pwa.pwa_data_term_static(A_dev, Vs[1], out_b, cuda_stream=stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                               # nothing was allocated on the device
    rec_a, rec_b = out_a.cpu().numpy(), out_b.cpu().numpy()
    _close(rec_a, refs[0], TOL[storage])
    _close(rec_b, refs[1], TOL[storage])
    # bitwise reproducible for a fixed shape, also with another call in between
    pwa.pwa_data_term_static(A_dev, Vs[0], out_b, cuda_stream=stream)
    assert np.array_equal(out_b.cpu().numpy(), rec_a)
    # and the definition itself
    L, T, bad = oracle.data_term(A, Vs[1])
    _close(rec_b, np.concatenate([[L, float(bad)], np.asarray(T).reshape(-1)]), TOL[storage])


def test_static_entry_point_limits_and_edge_cases(pwa):
    import torch
    n = pwa.PWA_STATIC_MAX_WAVES + 1
    A_dev = torch.zeros(10, n, 2, dtype=torch.float64, device="cuda")
    out = torch.zeros(2 + 2 * n, dtype=torch.float64, device="cuda")
    with pytest.raises(pwa.PwaError) as ei:
        pwa.pwa_data_term_static(A_dev, np.ones((n, 2)), out)
    assert ei.value.status == pwa.PWA_ERR_UNSUPPORTED and "PWA_STATIC_MAX_WAVES" in str(ei.value)
    n = 8
    A_dev = torch.randn(300, n, 2, dtype=torch.float64, device="cuda")
    out = torch.full((2 + 2 * n,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(pwa.PwaError):
        pwa.pwa_data_term_static(A_dev, np.full((n, 2), np.inf), out)
    with pytest.raises(pwa.PwaError):
        pwa.pwa_data_term_static(A_dev, np.ones((n, 2)), out, device=64)
    assert np.all(out.cpu().numpy() == 7.0)                                    # outputs untouched on errors
    pwa.pwa_data_term_static(A_dev, np.ones((n, 2)), out, n_events=0)          # empty sample: zeros
    assert np.all(out.cpu().numpy() == 0.0)
    A_dev[17] = 0.0                                                            # S = 0: ln 0 = -inf, counted
    pwa.pwa_data_term_static(A_dev, np.ones((n, 2)), out)
    rec = out.cpu().numpy()
    assert rec[0] == -np.inf and rec[1] == 1.0
