"""Event-sharded evaluation on the GPU with TWO processes.

Only one GPU is available, so both ranks create their own pwa context on cuda:0 (independent kernels: no rank's
kernel waits on the other's) and exchange through gloo.  Every product line of the N > 1 path runs: shard bounds,
upload of the rank's block, pwa_build_norm -> pwa_norm_sums -> all-gather -> pwa_combine_norm_host -> pwa_set_norm,
then pwa_data_term_enqueue -> all-gather -> pwa_assemble_host_shards.  Results: bitwise equal on both ranks, equal to
the oracle on ALL events at 1e-12 / 1e-6, and equal to a single-context evaluation at the same tolerance.
"""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _case(seed, N, Nacc, n, storage):
    rng = np.random.default_rng(seed)
    dt = np.float64 if storage == "f64" else np.float32
    A = (rng.normal(size=(N, n, 2)) * 0.35).astype(dt)
    B = (rng.normal(size=(Nacc, n, 2)) * 0.35).astype(dt)
    V = rng.normal(size=(3, n, 2))
    return A, B, V


def _worker(rank, ws, port, seed, N, Nacc, n, storage, out_dir):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    try:
        from paper_1108_5882_b200 import binding as pwa
        from paper_1108_5882_b200 import sharded
        torch.cuda.set_device(0)
        A, B, Vs = _case(seed, N, Nacc, n, storage)
        n_gen_total = Nacc + 11
        lo, hi = sharded.shard_bounds(N, rank, ws)
        mlo, mhi = sharded.shard_bounds(Nacc, rank, ws)
        glo, ghi = sharded.shard_bounds(n_gen_total, rank, ws)
        ctx = pwa.pwa_create(n, storage, 0, torch.cuda.current_stream().cuda_stream)
        try:
            pwa.pwa_upload_events(ctx, pwa.PWA_DATA, np.ascontiguousarray(A[lo:hi]))
            pwa.pwa_upload_events(ctx, pwa.PWA_MC, np.ascontiguousarray(B[mlo:mhi]), n_generated=ghi - glo)
            pwa.pwa_build_norm(ctx, want_M=False)
            M_all, n_gen = sharded.combine_norm(ctx)
            out_dev = torch.zeros(2 + 2 * n, dtype=torch.float64, device="cuda")
            res = [sharded.nll_grad(ctx, V, M_all, out_dev) for V in Vs]
            res2 = sharded.nll_grad(ctx, Vs[0], M_all, out_dev, likelihood=1, n_data_total=float(N))
            # the installed M serves the rank-local full evaluation too (M of ALL MC events, data of this rank)
            local = pwa.pwa_nll_grad(ctx, Vs[0])
            np.savez(os.path.join(out_dir, f"r{rank}.npz"), M=M_all, n_gen=n_gen,
                     nll=np.array([r[0] for r in res]), g=np.stack([r[1] for r in res]),
                     parts=np.stack([r[2] for r in res]), nll2=res2[0], g2=res2[1], local_norm=local[2][1],
                     launches=pwa.pwa_launch_count(ctx))
        finally:
            pwa.pwa_destroy(ctx)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("N,Nacc,n,storage", [(200_003, 100_001, 16, "f64"), (150_001, 80_003, 64, "f32"), (1001, 777, 5, "f64")])
def test_two_rank_sharded_gpu(tmp_path, oracle, N, Nacc, n, storage):
    import torch
    assert torch.cuda.is_available()
    from paper_1108_5882_b200 import binding as pwa
    ws, seed = 2, 1000 + n
    mp.spawn(_worker, args=(ws, _free_port(), seed, N, Nacc, n, storage, str(tmp_path)), nprocs=ws, join=True)
    r = [np.load(tmp_path / f"r{k}.npz") for k in range(ws)]
    for key in ("M", "nll", "g", "parts", "nll2", "g2"):                 # rank-ordered sums: the same bits on every rank
        assert np.array_equal(r[0][key], r[1][key]), key
    assert int(r[0]["n_gen"]) == Nacc + 11 and int(r[0]["launches"]) >= 5
    tol = 1e-12 if storage == "f64" else 1e-6
    A, B, Vs = _case(seed, N, Nacc, n, storage)
    M_o = oracle.norm_matrix(B, Nacc + 11)
    assert np.abs(r[0]["M"] - M_o).max() <= tol * np.abs(M_o).max()
    # single-context evaluation of ALL events (the N = 1 product path)
    ctx = pwa.pwa_create(n, storage)
    try:
        pwa.pwa_upload_events(ctx, pwa.PWA_DATA, A)
        pwa.pwa_upload_events(ctx, pwa.PWA_MC, B, n_generated=Nacc + 11)
        pwa.pwa_build_norm(ctx, want_M=False)
        single = [pwa.pwa_nll_grad(ctx, V) for V in Vs]
    finally:
        pwa.pwa_destroy(ctx)
    for i, V in enumerate(Vs):
        nll_o, g_o, parts_o, _ = oracle.nll_grad(A, M_o, V)
        for nll_r, g_r, parts_r in ((nll_o, g_o, parts_o), single[i]):
            assert abs(r[0]["nll"][i] - nll_r) <= tol * max(abs(nll_r), abs(parts_r[0]))
            assert np.abs(r[0]["g"][i] - g_r).max() <= tol * np.abs(g_r).max()
            assert np.abs(r[0]["parts"][i] - parts_r).max() <= tol * np.abs(parts_r).max()
    nll2_o, g2_o, _ = oracle.nll_grad_eq2(A, M_o, Vs[0])
    assert abs(r[0]["nll2"] - nll2_o) <= tol * max(abs(nll2_o), abs(oracle.data_term(A, Vs[0])[0]))
    assert np.abs(r[0]["g2"] - g2_o).max() <= tol * np.abs(g2_o).max()
    assert float(r[0]["local_norm"]) == pytest.approx(float(r[0]["parts"][0][1]), rel=1e-12)


def test_bench_two_ranks_on_one_gpu(tmp_path):
    """bench.py's N > 1 code (shard generation, combine_norm, the sharded step with its all-gather, max-over-ranks timing,
    the JSON line of rank 0) under torch.distributed.run with two ranks.  One GPU here, so the ranks share it and exchange
    through gloo (PWA_BENCH_BACKEND=gloo, a test switch: the driver's runs use nccl); sizes are reduced, the line is not a
    measurement."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, PWA_BENCH_BACKEND="gloo", MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "4", "--warmup", "3",
           "--n-data", "300000", "--n-mc", "400000"]
    r = subprocess.run(cmd, cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]                    # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["steps"] == 4
    assert d["value"] > 0 and d["e2e"]["value"] > 0 and d["gpu_launches"] >= 4
    assert d["config"]["n_data_per_gpu"] == 300000 and "event-sharded x2" in d["config"]["parallelism"]
    assert d["value"] == pytest.approx(2 * 300000 * d["config"]["n_waves"] / d["ms_per_step"] * 1e3, rel=1e-9)
    # the reference arm under the same launcher: rank 0 alone runs and prints, the other rank exits 0
    cmd_ref = cmd[:cmd.index(os.path.join(root, "bench.py")) + 1] + ["--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "3",
                                                                     "--n-data", "20000"]
    r = subprocess.run(cmd_ref, cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["impl"] == "reference"
