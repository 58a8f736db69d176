"""Event-sharded evaluation: world_size-2 gloo run on the CPU.

The per-shard data-term records and M sums are produced by the ORACLE here (no GPU in this
test); what is under test is the host-side N>1 logic of the product: shard bounds, the
all-gather plumbing of sharded.py, and the C ABI's host-only synthesis steps
(pwa_combine_norm_host, pwa_assemble_host_shards: shards added in rank order, bitwise identical
on all ranks).  The same path on a GPU with two processes: tests/test_gpu_sharded.py.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, ws, port, N, Nacc, n, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    try:
        from oracle import oracle
        from paper_1108_5882_b200 import binding as pwa
        from paper_1108_5882_b200 import sharded
        rng = np.random.default_rng(7)
        A = rng.normal(size=(N, n, 2)) * 0.35
        B = rng.normal(size=(Nacc, n, 2)) * 0.35
        V = rng.normal(size=(n, 2))
        n_gen_total = Nacc + 11
        lo, hi = sharded.shard_bounds(N, rank, ws)
        mlo, mhi = sharded.shard_bounds(Nacc, rank, ws)
        glo, ghi = sharded.shard_bounds(n_gen_total, rank, ws)
        # per-shard pieces (what pwa_build_norm / pwa_data_term_enqueue produce on a GPU rank)
        G_local = oracle.norm_matrix(B[mlo:mhi], 1)            # N_gen = 1: the plain sums B^H B (what pwa_norm_sums returns)
        L, T, bad = oracle.data_term(A[lo:hi], V)
        terms = torch.from_numpy(np.concatenate([[L, float(bad)], T.reshape(-1)]))
        M_all, n_gen = sharded.combine_norm_sums(G_local, ghi - glo)
        tot = sharded.gather_terms(terms)
        assert tot.shape == (ws, 2 + 2 * n)
        nll, g, parts = pwa.pwa_assemble_host_shards(tot, M_all, V)
        nll2, g2, parts2 = pwa.pwa_assemble_host_shards(tot, M_all, V, likelihood=1, n_data=float(N))
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), nll=nll, g=g, parts=parts, M=M_all, n_gen=n_gen, tot=tot,
                 nll2=nll2, g2=g2)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("N,Nacc,n", [(1001, 777, 5), (4096, 2049, 16)])
def test_two_rank_sharded_evaluation(tmp_path, oracle, N, Nacc, n):
    ws = 2
    mp.spawn(_worker, args=(ws, _free_port(), N, Nacc, n, str(tmp_path)), nprocs=ws, join=True)
    r = [np.load(tmp_path / f"r{k}.npz") for k in range(ws)]
    # every rank holds the bitwise identical result (rank-ordered sum)
    for key in ("nll", "g", "parts", "M", "tot", "nll2", "g2"):
        assert np.array_equal(r[0][key], r[1][key]), key
    rng = np.random.default_rng(7)
    A = rng.normal(size=(N, n, 2)) * 0.35
    B = rng.normal(size=(Nacc, n, 2)) * 0.35
    V = rng.normal(size=(n, 2))
    assert int(r[0]["n_gen"]) == Nacc + 11
    M_o = oracle.norm_matrix(B, Nacc + 11)
    assert np.abs(r[0]["M"] - M_o).max() <= 1e-13 * np.abs(M_o).max()
    nll_o, g_o, parts_o, _ = oracle.nll_grad(A, M_o, V)
    assert abs(r[0]["nll"] - nll_o) <= 1e-12 * max(abs(nll_o), abs(parts_o[0]))
    assert np.abs(r[0]["g"] - g_o).max() <= 1e-12 * np.abs(g_o).max()
    assert np.abs(r[0]["parts"] - parts_o).max() <= 1e-12 * np.abs(parts_o).max()
    nll2_o, g2_o, _ = oracle.nll_grad_eq2(A, M_o, V)
    assert abs(r[0]["nll2"] - nll2_o) <= 1e-12 * max(abs(nll2_o), abs(parts_o[0]))
    assert np.abs(r[0]["g2"] - g2_o).max() <= 1e-12 * np.abs(g2_o).max()


def test_shard_bounds_cover_exactly():
    from paper_1108_5882_b200 import sharded
    for n_events in (0, 1, 7, 8, 1000003):
        for ws in (1, 2, 3, 8):
            b = [sharded.shard_bounds(n_events, r, ws) for r in range(ws)]
            assert b[0][0] == 0 and b[-1][1] == n_events
            assert all(b[i][1] == b[i + 1][0] for i in range(ws - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1
