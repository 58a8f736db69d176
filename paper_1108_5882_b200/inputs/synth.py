"""Seeded synthetic workloads shaped like BASELINE.json configs[0..4].

This module only GENERATES INPUTS (kinematics, Breit-Wigner x spherical-harmonic amplitude
matrices, accepted-MC samples, evaluation points V).  It holds none of the likelihood /
gradient arithmetic, imports neither the CUDA binding nor the oracle, and is the only code
the two sides share: the identical arrays are handed to both (C15).

The paper's own workload (BES J/psi -> gamma K+K-) is not available and is
not reconstructed; these samples only stand in for its shape.
"""
import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "synth_gen.c")
LIB = os.path.join(HERE, "libpwa_synth.so")

DEFAULT_SEED = 20110829

# stream ids (C15): one base id per purpose; kinematic samples use base..base+3
S_DATA, S_MC, S_PILOT = 100, 200, 300
S_RES_M, S_RES_G, S_VTRUE, S_VEVAL, S_START = 400, 401, 500, 600, 700

_lib = None


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    subprocess.run(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-Wall",
                    "-o", LIB, SRC, "-lm"], check=True)
    return LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.pwa_gen_u64.restype = C.c_uint64
        _lib.pwa_gen_pilot_max.restype = C.c_double
        _lib.pwa_gen_accept.restype = C.c_int64
    return _lib


def _p(x):
    return x.ctypes.data_as(C.c_void_p)


def uniform(seed, stream, count, lo, hi, start=0):
    out = np.empty(count)
    lib().pwa_gen_uniform(C.c_uint64(seed), C.c_uint64(stream), C.c_int64(start),
                          C.c_int64(count), C.c_double(lo), C.c_double(hi), _p(out))
    return out


def cnormal(seed, stream, count, start=0):
    """[count, 2] float64: independent N(0,1) real and imaginary parts (C13)."""
    out = np.empty((count, 2))
    lib().pwa_gen_cnormal(C.c_uint64(seed), C.c_uint64(stream), C.c_int64(start),
                          C.c_int64(count), _p(out))
    return out


# (n_res, fixed resonances or None, N_data, N_acc, storage, use efficiency, factored)
_CFG = {
    0: dict(n_res=4, fixed=[(1.5, 0.1), (1.71, 0.14), (2.0, 0.2), (2.3, 0.25)],
            n_data=10_000, n_mc=50_000, storage="f64", eff=False, factored=False, evals=1),
    1: dict(n_res=8, fixed=None, n_data=100_000, n_mc=1_000_000, storage="f64", eff=True,
            factored=False, evals=100),
    2: dict(n_res=16, fixed=None, n_data=1_000_000, n_mc=10_000_000, storage="f32", eff=True,
            factored=False, evals=1000),
    3: dict(n_res=8, fixed=None, n_data=1_000_000, n_mc=4_000_000, storage="f64", eff=True,
            factored=True, evals=200, n_free=4),
    4: dict(n_res=32, fixed=None, n_data=5_000_000, n_mc=20_000_000, storage="f32", eff=True,
            factored=False, evals=300, K=64),
}


@dataclass
class Workload:
    cfg: int
    seed: int
    n: int
    n_res: int
    n_ang: int
    storage: str                 # "f64" | "f32": amplitude STORAGE type
    Mr: np.ndarray               # [n_res] resonance masses (GeV)
    Gr: np.ndarray               # [n_res] widths (GeV)
    res_of_wave: np.ndarray      # [n] int32
    ang_of_wave: np.ndarray      # [n] int32, index into yids
    yids: np.ndarray             # [n_ang] int32 angular structure ids (0:Y00 1:Y20 2:Y2+1 3:Y2-1)
    V_true: np.ndarray           # [n, 2]
    n_data: int
    n_acc: int
    n_gen: int
    kin_data: tuple = field(repr=False, default=None)   # (m, cos, phi)
    kin_mc: tuple = field(repr=False, default=None)
    A_data: Optional[np.ndarray] = field(repr=False, default=None)   # [N, n, 2]
    A_mc: Optional[np.ndarray] = field(repr=False, default=None)
    Z_data: Optional[np.ndarray] = field(repr=False, default=None)   # [N, n_ang, 2]
    Z_mc: Optional[np.ndarray] = field(repr=False, default=None)
    n_free: int = 0
    K: int = 1
    evals: int = 1
    i_max: float = 0.0
    n_over: int = 0

    @property
    def np_dtype(self):
        return np.float64 if self.storage == "f64" else np.float32

    @property
    def yid_of_wave(self):
        return np.ascontiguousarray(self.yids[self.ang_of_wave], dtype=np.int32)

    @property
    def mass_data(self):
        return self.kin_data[0]

    @property
    def mass_mc(self):
        return self.kin_mc[0]


def _model_args(w):
    return (C.c_int(w.n_res), _p(w.Mr), _p(w.Gr), C.c_int(w.n), _p(w.res_of_wave),
            _p(w.yid_of_wave))


def amplitudes(w: Workload, kin, storage=None):
    """Full [N, n, 2] amplitude matrix at the workload's (Mr, Gr)."""
    m, c, p = kin
    dt = 0 if (storage or w.storage) == "f64" else 1
    out = np.empty((m.shape[0], w.n, 2), dtype=np.float64 if dt == 0 else np.float32)
    yw = w.yid_of_wave
    lib().pwa_gen_amplitudes(_p(m), _p(c), _p(p), C.c_int64(m.shape[0]), C.c_int(w.n_res),
                             _p(w.Mr), _p(w.Gr), C.c_int(w.n), _p(w.res_of_wave), _p(yw),
                             C.c_int(dt), _p(out))
    return out


def angular(w: Workload, kin, storage=None):
    """[N, n_ang, 2] angular factors Z (factored upload)."""
    m, c, p = kin
    dt = 0 if (storage or w.storage) == "f64" else 1
    out = np.empty((m.shape[0], w.n_ang, 2), dtype=np.float64 if dt == 0 else np.float32)
    lib().pwa_gen_angular(_p(c), _p(p), C.c_int64(m.shape[0]), C.c_int(w.n_ang), _p(w.yids),
                          C.c_int(dt), _p(out))
    return out


def _accept(w, seed, s0, n_want, mode, i_max, V):
    m, c, p = np.empty(n_want), np.empty(n_want), np.empty(n_want)
    drawn, over = C.c_int64(0), C.c_int64(0)
    yw = w.yid_of_wave
    got = lib().pwa_gen_accept(C.c_uint64(seed), C.c_uint64(s0), C.c_int64(n_want), C.c_int(mode),
                               C.c_double(i_max), C.c_int(w.n_res), _p(w.Mr), _p(w.Gr),
                               C.c_int(w.n), _p(w.res_of_wave), _p(yw), _p(V),
                               _p(m), _p(c), _p(p), C.byref(drawn), C.byref(over))
    assert got == n_want
    return (m, c, p), int(drawn.value), int(over.value)


def make_workload(cfg: int, seed: int = DEFAULT_SEED, n_data: Optional[int] = None,
                  n_mc: Optional[int] = None, storage: Optional[str] = None,
                  want_data: bool = True, want_mc: bool = True,
                  full_amplitudes: bool = True, shard: int = 0) -> Workload:
    """Build configs[cfg] (optionally with reduced event counts for CPU-side tests).

    want_data / want_mc = False skip generating that sample (bench legs that need one only).
    full_amplitudes=False skips the [N, n, 2] matrices for a factored workload.
    shard: index of an event-sharded rank (0..23).  The model (resonances, V_true, I_max) is
    the same for every shard; only the candidate streams of the data and MC kinematics differ,
    so shards are disjoint, independent samples of the same distribution.
    """
    if not 0 <= shard < 24:
        raise ValueError("shard must be in [0, 24)")
    spec = _CFG[cfg]
    n_res = spec["n_res"]
    if spec["fixed"] is not None:
        Mr = np.array([x[0] for x in spec["fixed"]])
        Gr = np.array([x[1] for x in spec["fixed"]])
        n = 4
        res_of_wave = np.arange(4, dtype=np.int32)
        yids = np.array([0, 1, 2], dtype=np.int32)
        ang_of_wave = np.array([0, 0, 1, 2], dtype=np.int32)          # C5
    else:
        Mr = uniform(seed, S_RES_M, n_res, 1.2, 2.8)
        Gr = uniform(seed, S_RES_G, n_res, 0.05, 0.3)
        n = 2 * n_res
        res_of_wave = (np.arange(n) // 2).astype(np.int32)
        yids = np.array([0, 2], dtype=np.int32)
        ang_of_wave = (np.arange(n) % 2).astype(np.int32)            # C5
    V_true = cnormal(seed, S_VTRUE, n)
    w = Workload(cfg=cfg, seed=seed, n=n, n_res=n_res, n_ang=len(yids),
                 storage=storage or spec["storage"], Mr=Mr, Gr=Gr, res_of_wave=res_of_wave,
                 ang_of_wave=ang_of_wave, yids=yids, V_true=V_true,
                 n_data=int(n_data or spec["n_data"]), n_acc=int(n_mc or spec["n_mc"]), n_gen=0,
                 n_free=spec.get("n_free", 0), K=spec.get("K", 1), evals=spec["evals"])
    eff = 1 if spec["eff"] else 0
    yw = w.yid_of_wave
    if want_data:
        pilot = lib().pwa_gen_pilot_max(C.c_uint64(seed), C.c_uint64(S_PILOT), C.c_int64(200_000),
                                        C.c_int(eff), C.c_int(n_res), _p(Mr), _p(Gr), C.c_int(n),
                                        _p(res_of_wave), _p(yw), _p(V_true))
        w.i_max = 1.5 * float(pilot)                                  # C11
        w.kin_data, _, w.n_over = _accept(w, seed, S_DATA + 4 * shard, w.n_data, 2 | eff, w.i_max, V_true)
    if want_mc:
        w.kin_mc, w.n_gen, _ = _accept(w, seed, S_MC + 4 * shard, w.n_acc, eff, 1.0, V_true)   # C9
    factored = spec["factored"]
    if factored:
        if want_data:
            w.Z_data = angular(w, w.kin_data)
        if want_mc:
            w.Z_mc = angular(w, w.kin_mc)
    if (not factored) or full_amplitudes:
        if want_data:
            w.A_data = amplitudes(w, w.kin_data)
        if want_mc:
            w.A_mc = amplitudes(w, w.kin_mc)
    return w


def eval_points(w: Workload, count: int, stream: int = S_VEVAL) -> np.ndarray:
    """[count, n, 2] random evaluation points / starting vectors, V ~ CN (C13)."""
    return cnormal(w.seed, stream, count * w.n).reshape(count, w.n, 2)


def floating_start(w: Workload):
    """cfg 3 fit start: free (M_r, G_r) = truth * (1 + 0.02 N(0,1))."""
    z = cnormal(w.seed, S_START, w.n_res)
    Mr, Gr = w.Mr.copy(), w.Gr.copy()
    Mr[: w.n_free] *= 1.0 + 0.02 * z[: w.n_free, 0]
    Gr[: w.n_free] *= 1.0 + 0.02 * z[: w.n_free, 1]
    return Mr, Gr
