"""Event-sharded evaluation: world_size-2 gloo run on the CPU.

The per-shard data-term records and M matrices are produced by the ORACLE here (no GPU in this
test); what is under test is the host-side N>1 logic of the product: shard bounds, the
rank-ordered sum (bitwise identical on all ranks), the N_gen-weighted M combination and the
final assembly through the C ABI's host-only pwa_assemble_host.
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
        M_local = oracle.norm_matrix(B[mlo:mhi], ghi - glo)
        L, T, bad = oracle.data_term(A[lo:hi], V)
        terms = torch.from_numpy(np.concatenate([[L, float(bad)], T.reshape(-1)]))
        M_all, n_gen = sharded.combine_norm(M_local, ghi - glo)
        tot = sharded.reduce_terms(terms).numpy()
        nll, g, parts = pwa.pwa_assemble_host(tot[0], tot[2:].reshape(n, 2), M_all, V)
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), nll=nll, g=g, parts=parts, M=M_all, n_gen=n_gen, tot=tot)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("N,Nacc,n", [(1001, 777, 5), (4096, 2049, 16)])
def test_two_rank_sharded_evaluation(tmp_path, oracle, N, Nacc, n):
    ws = 2
    mp.spawn(_worker, args=(ws, _free_port(), N, Nacc, n, str(tmp_path)), nprocs=ws, join=True)
    r = [np.load(tmp_path / f"r{k}.npz") for k in range(ws)]
    # every rank holds the bitwise identical result (rank-ordered sum)
    for key in ("nll", "g", "parts", "M", "tot"):
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


def test_shard_bounds_cover_exactly():
    from paper_1108_5882_b200 import sharded
    for n_events in (0, 1, 7, 8, 1000003):
        for ws in (1, 2, 3, 8):
            b = [sharded.shard_bounds(n_events, r, ws) for r in range(ws)]
            assert b[0][0] == 0 and b[-1][1] == n_events
            assert all(b[i][1] == b[i + 1][0] for i in range(ws - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1
