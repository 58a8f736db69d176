"""Pins of the CPU oracle (oracle/pwa_oracle.c) against what the paper and mathematics fix.

No GPU.  The paper prints no worked numbers (P0), so each pin is a closed form, an
invariant, an exact-rational brute force, or a reduction to a numpy/BLAS routine, chosen so
that a dropped term, wrong sign/conjugation, factor 2 or transposed index fails one of them.
Pin numbers follow SURVEY.md section 8(c) / DESIGN.md section 5.
P:n = /root/reference/PAPER.md line n (cited, never read at run time).
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def cplx(x):
    x = np.asarray(x)
    return x[..., 0] + 1j * x[..., 1]


def ri(z):
    z = np.asarray(z)
    return np.ascontiguousarray(np.stack([z.real, z.imag], axis=-1))


def rand_amps(rng, N, n, scale=0.35):
    return rng.normal(size=(N, n, 2)) * scale


def full_eval(oracle, A, B, n_gen, V):
    M = oracle.norm_matrix(B, n_gen)
    return oracle.nll_grad(A, M, V), M


# ---------------------------------------------------------------- P0 / storage remark
def test_paper_storage_remark():
    """n^2 fp32 reals per event: 1e6 * 20^2 * 4 B = 1.49 GiB ~ '1.5 GB'."""
    kv = {}
    for line in open(os.path.join(GOLD, "paper_storage_remark.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        kv[k] = float(v)
    gib = kv["events"] * kv["waves"] ** 2 * kv["bytes_per_real"] / 2 ** 30
    assert abs(gib - kv["quoted_gib"]) < 0.05
    # the streamed N x n complex matrix of this build is n/2 times smaller in fp32
    assert kv["events"] * kv["waves"] * 8 * (kv["waves"] / 2) == kv["events"] * kv["waves"] ** 2 * 4


# ---------------------------------------------------------------- P1 single-wave closed form
def test_p1_single_wave_constant_amplitudes(oracle):
    N, Nacc, Ngen = 1000, 700, 1000
    A = np.zeros((N, 1, 2)); A[..., 0] = 1.0
    B = np.zeros((Nacc, 1, 2)); B[..., 0] = 1.0
    V = np.array([[0.8, -1.3]])
    (nll, g, parts, bad), M = full_eval(oracle, A, B, Ngen, V)
    v2 = 0.8 ** 2 + 1.3 ** 2
    lnL = N * math.log(v2) - v2 * Nacc / Ngen
    assert bad == 0
    assert nll == pytest.approx(-lnL, rel=1e-15)
    assert cplx(M)[0, 0] == pytest.approx(Nacc / Ngen, rel=1e-15)
    gexp = -2 * N * cplx(V)[0] / v2 + 2 * (Nacc / Ngen) * cplx(V)[0]
    assert cplx(g)[0] == pytest.approx(gexp, rel=1e-14)
    # stationary point of eq. 3 at |V|^2 = N / M11 (P7 corollary): gradient vanishes there
    Vs = np.array([[math.sqrt(N / (Nacc / Ngen)), 0.0]])
    nll_s, g_s, parts_s, _ = oracle.nll_grad(A, M, Vs)
    assert np.abs(g_s).max() < 1e-10
    assert parts_s[1] == pytest.approx(N, rel=1e-14)


def test_p1_single_wave_random_amplitudes(oracle):
    rng = np.random.default_rng(11)
    N, Nacc, Ngen = 513, 901, 1300
    A, B = rand_amps(rng, N, 1), rand_amps(rng, Nacc, 1)
    V = np.array([[-0.4, 0.9]])
    (nll, g, parts, _), M = full_eval(oracle, A, B, Ngen, V)
    v2 = float(np.abs(cplx(V)[0]) ** 2)
    M11 = float((np.abs(cplx(B)[:, 0]) ** 2).sum() / Ngen)
    lnL = N * math.log(v2) + float(np.log(np.abs(cplx(A)[:, 0]) ** 2).sum()) - v2 * M11
    assert nll == pytest.approx(-lnL, rel=1e-13)
    gexp = -2 * N * cplx(V)[0] / v2 + 2 * M11 * cplx(V)[0]
    assert cplx(g)[0] == pytest.approx(gexp, rel=1e-12)


# ---------------------------------------------------------------- P2 global phase
def test_p2_global_phase(oracle):
    rng = np.random.default_rng(2)
    n = 5
    A, B = rand_amps(rng, 400, n), rand_amps(rng, 700, n)
    V = rng.normal(size=(n, 2))
    (nll, g, parts, _), M = full_eval(oracle, A, B, 900, V)
    for th in (0.3, 1.7, math.pi):
        Vr = ri(np.exp(1j * th) * cplx(V))
        nll2, g2, parts2, _ = oracle.nll_grad(A, M, Vr)
        assert nll2 == pytest.approx(nll, rel=1e-13)
        assert np.allclose(cplx(g2), np.exp(1j * th) * cplx(g), rtol=1e-11, atol=1e-11 * np.abs(g).max())
    # infinitesimal form, separately for data and norm terms: Im(V^H g) = 0
    L, T, _ = oracle.data_term(A, V)
    g_data = 2 * np.conj(cplx(T))
    Nv, gN = oracle.norm_explicit(B, 900, V)
    Vc = cplx(V)
    assert abs(np.imag(np.vdot(Vc, g_data))) < 1e-10 * np.abs(g_data).max()
    assert abs(np.imag(np.vdot(Vc, cplx(gN)))) < 1e-12 * np.abs(gN).max()


# ---------------------------------------------------------------- P3 M Hermitian PSD
def test_p3_norm_matrix_hermitian_psd(oracle):
    rng = np.random.default_rng(3)
    n = 6
    B = rand_amps(rng, 2000, n)
    M = cplx(oracle.norm_matrix(B, 2500))
    assert np.allclose(M, M.conj().T, rtol=0, atol=1e-16)
    assert np.all(M.diagonal().real >= 0) and np.abs(M.diagonal().imag).max() == 0.0
    ev = np.linalg.eigvalsh(M)
    assert ev.min() >= -1e-13 * np.trace(M).real
    for _ in range(5):
        x = rng.normal(size=n) + 1j * rng.normal(size=n)
        assert np.vdot(x, M @ x).real >= 0


# ---------------------------------------------------------------- P4 M <-> explicit MC sum (C1)
def test_p4_norm_index_convention(oracle):
    rng = np.random.default_rng(4)
    n, Ngen = 4, 1234
    B = rand_amps(rng, 1000, n)
    V = rng.normal(size=(n, 2))
    M = cplx(oracle.norm_matrix(B, Ngen))
    Vc = cplx(V)
    Nprime, gN = oracle.norm_explicit(B, Ngen, V)
    # independent third opinion of the explicit sum
    Nnp = float((np.abs(cplx(B) @ Vc) ** 2).sum() / Ngen)
    assert Nprime == pytest.approx(Nnp, rel=1e-13)
    assert np.vdot(Vc, M @ Vc).real == pytest.approx(Nprime, rel=1e-13)
    assert np.allclose(2 * M @ Vc, cplx(gN), rtol=1e-12)
    # the transposed pairing V^T M conj(V) (eq. 3's bracket read literally, C1) is a different number
    wrong = (Vc @ M @ Vc.conj()).real
    assert abs(wrong - Nprime) > 1e-3 * abs(Nprime)
    # assemble() uses the same convention
    nll, g, parts = oracle.assemble(0.0, np.zeros((n, 2)), ri(M), V)
    assert parts[1] == pytest.approx(Nprime, rel=1e-13)
    assert np.allclose(cplx(g), cplx(gN), rtol=1e-12)


# ---------------------------------------------------------------- P5 gradient vs differences
@pytest.mark.parametrize("n", [1, 3, 8])
def test_p5_gradient_central_differences(oracle, n):
    rng = np.random.default_rng(50 + n)
    A, B = rand_amps(rng, 300, n), rand_amps(rng, 500, n)
    V = rng.normal(size=(n, 2))
    (nll, g, parts, _), M = full_eval(oracle, A, B, 800, V)
    num = np.zeros_like(V)
    for a in range(n):
        for c in range(2):
            h = 1e-6 * max(1.0, abs(V[a, c]))
            Vp, Vm = V.copy(), V.copy()
            Vp[a, c] += h; Vm[a, c] -= h
            fp = oracle.nll_grad(A, M, Vp)[0]
            fm = oracle.nll_grad(A, M, Vm)[0]
            num[a, c] = (fp - fm) / (2 * h)
    assert np.abs(num - g).max() <= 2e-8 * np.abs(g).max()


# ---------------------------------------------------------------- P6 + brute force (exact rationals)
def _load_tiny():
    A, V, ngen = [], None, None
    for line in open(os.path.join(GOLD, "tiny_dyadic_case.txt")):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] == "A":
            A.append([float(x) for x in t[1:]])
        elif t[0] == "V":
            V = [float(x) for x in t[1:]]
        elif t[0] == "NGEN":
            ngen = int(t[1])
    return np.array(A).reshape(3, 2, 2), np.array(V).reshape(2, 2), ngen


def _fc(re, im):
    return (Fraction(re), Fraction(im))


def _fmul(x, y):
    return (x[0] * y[0] - x[1] * y[1], x[0] * y[1] + x[1] * y[0])


def _fconj(x):
    return (x[0], -x[1])


def test_p6_eq1_equals_eq3_and_exact_bruteforce(oracle):
    """eq. 1 == eq. 3's double sum with zero imaginary part, checked in exact
    rational arithmetic; L_data, T, M, Norm, gradient brute-forced from the definitions."""
    A, V, ngen = _load_tiny()
    N, n = A.shape[0], A.shape[1]
    Af = [[_fc(A[i, a, 0], A[i, a, 1]) for a in range(n)] for i in range(N)]
    Vf = [_fc(V[a, 0], V[a, 1]) for a in range(n)]
    L_exact, T_exact = 0.0, [(Fraction(0), Fraction(0)) for _ in range(n)]
    for i in range(N):
        S = (Fraction(0), Fraction(0))
        for a in range(n):
            p = _fmul(Vf[a], Af[i][a]); S = (S[0] + p[0], S[1] + p[1])
        I1 = S[0] ** 2 + S[1] ** 2
        dbl = (Fraction(0), Fraction(0))
        for a in range(n):
            for b in range(n):
                t = _fmul(_fmul(Vf[a], _fconj(Vf[b])), _fmul(Af[i][a], _fconj(Af[i][b])))
                dbl = (dbl[0] + t[0], dbl[1] + t[1])
        assert dbl[1] == 0 and dbl[0] == I1                    # exact identity
        # oracle's two forms (all products exact in binary floating point for this fixture)
        assert oracle.intensity_eq1(A[i], V) == float(I1)
        e3 = oracle.intensity_eq3(A[i], V)
        assert e3.real == float(I1) and e3.imag == 0.0
        L_exact += math.log(float(I1))
        for a in range(n):   # A/S = A conj(S)/I
            q = _fmul(Af[i][a], _fconj(S))
            T_exact[a] = (T_exact[a][0] + q[0] / I1, T_exact[a][1] + q[1] / I1)
    L, T, bad = oracle.data_term(A, V)
    assert bad == 0 and L == pytest.approx(L_exact, rel=1e-15)
    for a in range(n):
        assert T[a, 0] == pytest.approx(float(T_exact[a][0]), rel=1e-15)
        assert T[a, 1] == pytest.approx(float(T_exact[a][1]), rel=1e-15)
    # use the same 3 events as "MC": M_ab = sum_j conj(B_ja) B_jb / ngen exactly
    M = oracle.norm_matrix(A, ngen)
    for a in range(n):
        for b in range(n):
            acc = (Fraction(0), Fraction(0))
            for j in range(N):
                t = _fmul(_fconj(Af[j][a]), Af[j][b]); acc = (acc[0] + t[0], acc[1] + t[1])
            assert M[a, b, 0] == float(acc[0] / ngen) and M[a, b, 1] == float(acc[1] / ngen)
    # Norm = (1/ngen) sum_j |S_j|^2 exactly, gradient = -2 conj(T) + (2/ngen) sum_j conj(B_ja) S_j
    Nx = Fraction(0)
    gN = [(Fraction(0), Fraction(0)) for _ in range(n)]
    for j in range(N):
        S = (Fraction(0), Fraction(0))
        for a in range(n):
            p = _fmul(Vf[a], Af[j][a]); S = (S[0] + p[0], S[1] + p[1])
        Nx += S[0] ** 2 + S[1] ** 2
        for a in range(n):
            t = _fmul(_fconj(Af[j][a]), S); gN[a] = (gN[a][0] + 2 * t[0] / ngen, gN[a][1] + 2 * t[1] / ngen)
    nll, g, parts, _ = oracle.nll_grad(A, M, V)
    assert parts[1] == pytest.approx(float(Nx / ngen), rel=1e-15)
    assert nll == pytest.approx(-(L_exact - float(Nx / ngen)), rel=1e-14)
    for a in range(n):
        assert g[a, 0] == pytest.approx(-2 * float(T_exact[a][0]) + float(gN[a][0]), rel=1e-13)
        assert g[a, 1] == pytest.approx(+2 * float(T_exact[a][1]) + float(gN[a][1]), rel=1e-13)


# ---------------------------------------------------------------- P7 Euler / scale identity
def test_p7_euler_identity(oracle):
    rng = np.random.default_rng(7)
    n, N = 7, 1500
    A, B = rand_amps(rng, N, n), rand_amps(rng, 900, n)
    V = rng.normal(size=(n, 2))
    L, T, _ = oracle.data_term(A, V)
    assert np.sum(cplx(V) * cplx(T)) == pytest.approx(N, rel=1e-13)       # sum_a V_a T_a = N exactly
    Nv, gN = oracle.norm_explicit(B, 1000, V)
    assert np.vdot(cplx(V), cplx(gN)).real == pytest.approx(2 * Nv, rel=1e-13)
    # scaling law: L(sV) = L(V) + N ln s^2 ; Norm(sV) = s^2 Norm(V)
    s = 1.7
    L2, _, _ = oracle.data_term(A, s * V)
    assert L2 == pytest.approx(L + N * math.log(s * s), rel=1e-13)
    assert oracle.norm_explicit(B, 1000, s * V)[0] == pytest.approx(s * s * Nv, rel=1e-13)


# ---------------------------------------------------------------- P8 numpy / BLAS third opinion
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_p8_reduces_to_blas(oracle, dtype):
    rng = np.random.default_rng(8)
    n, N, Nacc, Ngen = 12, 3000, 4000, 5000
    A = rand_amps(rng, N, n).astype(dtype)
    B = rand_amps(rng, Nacc, n).astype(dtype)
    V = rng.normal(size=(n, 2))
    Ac, Bc, Vc = cplx(A.astype(np.float64)), cplx(B.astype(np.float64)), cplx(V)
    M = oracle.norm_matrix(B, Ngen)
    assert np.allclose(cplx(M), Bc.conj().T @ Bc / Ngen, rtol=1e-13, atol=1e-15)
    S = Ac @ Vc
    L, T, _ = oracle.data_term(A, V)
    assert L == pytest.approx(np.log(np.abs(S) ** 2).sum(), rel=1e-13)
    assert np.allclose(cplx(T), (Ac / S[:, None]).sum(0), rtol=1e-12, atol=1e-12 * np.abs(T).max())
    # batched = loop (step 9)
    Vk = rng.normal(size=(3, n, 2))
    nllk, gk, partsk, _ = oracle.nll_grad_batch(A, M, Vk)
    Sk = Ac @ cplx(Vk).T
    assert np.allclose(partsk[:, 0], np.log(np.abs(Sk) ** 2).sum(0), rtol=1e-13)
    for k in range(3):
        one = oracle.nll_grad(A, M, Vk[k])
        assert one[0] == nllk[k] and np.array_equal(one[1], gk[k])


def test_fp32_storage_is_exact_widening(oracle):
    """C16: fp32-stored amplitudes are widened exactly; same bits as the widened fp64 array."""
    rng = np.random.default_rng(16)
    A32 = rand_amps(rng, 700, 5).astype(np.float32)
    B32 = rand_amps(rng, 900, 5).astype(np.float32)
    V = rng.normal(size=(5, 2))
    M32, M64 = oracle.norm_matrix(B32, 1000), oracle.norm_matrix(B32.astype(np.float64), 1000)
    assert np.array_equal(M32, M64)
    r32, r64 = oracle.nll_grad(A32, M32, V), oracle.nll_grad(A32.astype(np.float64), M64, V)
    assert r32[0] == r64[0] and np.array_equal(r32[1], r64[1])


# ---------------------------------------------------------------- P9 structural invariances
def test_p9_invariances(oracle):
    rng = np.random.default_rng(9)
    n, N = 4, 2000
    A = rand_amps(rng, N, n)
    V = rng.normal(size=(n, 2))
    L, T, _ = oracle.data_term(A, V)
    # permutation
    perm = rng.permutation(N)
    Lp, Tp, _ = oracle.data_term(A[perm], V)
    assert Lp == pytest.approx(L, rel=1e-14) and np.allclose(Tp, T, rtol=1e-12, atol=1e-13)
    # duplication doubles L and T
    Ld, Td, _ = oracle.data_term(np.concatenate([A, A]), V)
    assert Ld == pytest.approx(2 * L, rel=1e-14) and np.allclose(Td, 2 * T, rtol=1e-12, atol=1e-13)
    # A -> cA: S -> cS, so L + N ln|c|^2 and T = sum A/S is UNCHANGED
    # (SURVEY.md P9 says 'T/c'; that is a slip: the c cancels in A_ia / S_i)
    c = 0.7 - 1.9j
    Lc, Tc, _ = oracle.data_term(ri(c * cplx(A)), V)
    assert Lc == pytest.approx(L + N * math.log(abs(c) ** 2), rel=1e-13)
    assert np.allclose(cplx(Tc), cplx(T), rtol=1e-11, atol=1e-12)
    # two identical columns -> depends on V_0 + V_1 only
    A2 = A.copy(); A2[:, 1] = A2[:, 0]
    V2 = V.copy(); V2[0] = V[0] + V[1] - np.array([0.3, -0.2]); V2[1] = np.array([0.3, -0.2])
    assert oracle.data_term(A2, V2)[0] == pytest.approx(oracle.data_term(A2, V)[0], rel=1e-13)
    # thread-count independence to rounding
    from oracle import oracle as o
    nt = o.threads()
    o.set_threads(1)
    L1, T1, _ = o.data_term(A, V)
    o.set_threads(nt)
    assert L1 == pytest.approx(L, rel=1e-15) and np.allclose(T1, T, rtol=1e-14, atol=1e-15)


# ---------------------------------------------------------------- P10 Breit-Wigner (C3)
def test_p10_breit_wigner(oracle):
    M, G = 1.71, 0.14
    assert oracle.bw(M, M, G) == pytest.approx(1j / (M * G), rel=1e-15)       # pure imaginary on the pole
    for m in (1.0, 1.6, 1.71, 2.4):
        bw = oracle.bw(m, M, G)
        assert bw == pytest.approx(1.0 / (M * M - m * m - 1j * M * G), rel=1e-15)
        assert abs(bw) ** 2 == pytest.approx(1.0 / ((M * M - m * m) ** 2 + (M * G) ** 2), rel=1e-14)
    # half maximum of |BW|^2 at m^2 = M^2 +- M G
    peak = abs(oracle.bw(M, M, G)) ** 2
    for sgn in (+1, -1):
        m = math.sqrt(M * M + sgn * M * G)
        assert abs(oracle.bw(m, M, G)) ** 2 == pytest.approx(peak / 2, rel=1e-13)
    # derivatives vs central differences
    for m in (1.2, 1.7, 2.2):
        dM, dG = oracle.bw_deriv(m, M, G)
        h = 1e-6
        nM = (oracle.bw(m, M + h, G) - oracle.bw(m, M - h, G)) / (2 * h)
        nG = (oracle.bw(m, M, G + h) - oracle.bw(m, M, G - h)) / (2 * h)
        assert dM == pytest.approx(nM, rel=1e-7) and dG == pytest.approx(nG, rel=1e-7)


def test_factored_expansion_matches_generator(oracle, synth):
    """Oracle step 1 (A = BW * Z, own BW code) vs the generator's own line-shape code."""
    w = synth.make_workload(3, n_data=2000, n_mc=3000)
    A = oracle.expand_factored(w.mass_data, w.Z_data, w.res_of_wave, w.ang_of_wave, w.Mr, w.Gr)
    assert np.allclose(A, w.A_data, rtol=1e-13, atol=1e-15)
    # explicit complex formula, third opinion
    m = w.mass_data[:, None]
    bw = 1.0 / (w.Mr[None, :] ** 2 - m ** 2 - 1j * w.Mr[None, :] * w.Gr[None, :])
    ref = bw[:, w.res_of_wave] * cplx(w.Z_data)[:, w.ang_of_wave]
    assert np.allclose(cplx(A), ref, rtol=1e-13, atol=1e-15)


def test_res_grad_vs_differences(oracle, synth):
    """Reading A9: d L_data / d(M_r, G_r) and d Norm / d(M_r, G_r) vs central differences."""
    w = synth.make_workload(3, n_data=1500, n_mc=2500)
    V = synth.eval_points(w, 1)[0]
    Mr, Gr = w.Mr.copy(), w.Gr.copy()
    dM, dG = oracle.res_grad(w.mass_data, w.Z_data, w.res_of_wave, w.ang_of_wave, Mr, Gr, V, 0)
    nM, nG = oracle.res_grad(w.mass_mc, w.Z_mc, w.res_of_wave, w.ang_of_wave, Mr, Gr, V, 1, w.n_gen)

    def L_of(Mx, Gx):
        A = oracle.expand_factored(w.mass_data, w.Z_data, w.res_of_wave, w.ang_of_wave, Mx, Gx)
        return oracle.data_term(A, V)[0]

    def N_of(Mx, Gx):
        B = oracle.expand_factored(w.mass_mc, w.Z_mc, w.res_of_wave, w.ang_of_wave, Mx, Gx)
        return oracle.norm_explicit(B, w.n_gen, V)[0]

    h = 1e-6
    for r in range(w.n_res):
        for which, (aL, aN) in enumerate(((dM, nM), (dG, nG))):
            P, Q = (Mr.copy(), Gr.copy()), (Mr.copy(), Gr.copy())
            P[which][r] += h; Q[which][r] -= h
            numL = (L_of(*P) - L_of(*Q)) / (2 * h)
            numN = (N_of(*P) - N_of(*Q)) / (2 * h)
            assert aL[r] == pytest.approx(numL, rel=2e-6, abs=1e-6 * np.abs(dM).max())
            assert aN[r] == pytest.approx(numN, rel=2e-6, abs=1e-6 * max(np.abs(nM).max(), 1e-12))


# ---------------------------------------------------------------- C14 non-finite propagation
def test_c14_zero_intensity(oracle):
    A = np.zeros((3, 2, 2)); A[0, 0, 0] = 1.0; A[2, 1, 1] = 0.5     # event 1 has S = 0
    V = np.array([[1.0, 0.0], [0.0, 1.0]])
    L, T, bad = oracle.data_term(A, V)
    assert bad == 1 and L == -math.inf


# ---------------------------------------------------------------- configs 0/1 sanity (P11, P12-lite)
def test_cfg0_sanity_and_orthogonality(oracle, synth):
    w = synth.make_workload(0)
    assert w.n == 4 and w.n_gen == w.n_acc == 50_000 and w.n_over == 0
    # P11: over a flat full-acceptance MC, 4 pi <conj(Z^s) Z^s'> -> delta_ss'
    Z = cplx(synth.angular(w, w.kin_mc))
    G = 4 * math.pi * (Z.conj().T @ Z) / Z.shape[0]
    assert np.abs(G - np.eye(3)).max() < 5.0 / math.sqrt(Z.shape[0])
    M = oracle.norm_matrix(w.A_mc, w.n_gen)
    nll, g, parts, bad = oracle.nll_grad(w.A_data, M, w.V_true)
    assert bad == 0 and np.isfinite(nll)
    # the data were generated from V_true: lnL at truth beats a random point after optimal rescaling
    # (scale-profiled: max_s lnL(sV) = L - N ln(Norm/N) - N), P7
    def profiled(V):
        _, _, p, _ = oracle.nll_grad(w.A_data, M, V)
        return p[0] - w.n_data * math.log(p[1] / w.n_data) - w.n_data
    assert profiled(w.V_true) > profiled(synth.eval_points(w, 1)[0])


def test_cfg1_generator_recipe(synth):
    w = synth.make_workload(1, n_data=20_000, n_mc=50_000)
    assert w.n == 16 and w.n_res == 8 and w.storage == "f64"
    assert 1.2 <= w.Mr.min() and w.Mr.max() <= 2.8 and 0.05 <= w.Gr.min() and w.Gr.max() <= 0.3
    assert abs(w.n_acc / w.n_gen - 0.7) < 0.01            # C9: mean efficiency 0.700
    m, c, p = w.kin_mc
    assert m.min() >= 0.988 and m.max() <= 3.0 and abs(c).max() <= 1 and 0 <= p.min() and p.max() < 2 * math.pi
    # determinism / order independence of the counter-based RNG
    w2 = synth.make_workload(1, n_data=20_000, n_mc=50_000)
    assert np.array_equal(w.A_data, w2.A_data) and w.n_gen == w2.n_gen
    # a shorter request is a prefix of a longer one
    w3 = synth.make_workload(1, n_data=5_000, n_mc=10_000)
    assert np.array_equal(w3.A_data, w.A_data[:5000]) and np.array_equal(w3.A_mc, w.A_mc[:10000])


# ---------------------------------------------------------------- P13 eq. 2 (normalised) form, P14 polar parameters
def test_p13_eq2_form(oracle):
    """eq. 2 with the MC integral of P:35: nll2 = -L_data + N ln Norm.
    (a) independent of the overall scale of V (eq. 2 is a ratio); (b) gradient vs central
    differences; (c) at a V with Norm(V) = N it equals eq. 3 up to the constant N ln N - N and has
    the SAME gradient; (d) numpy restatement of the definition."""
    rng = np.random.default_rng(13)
    N, Nacc, n = 400, 700, 5
    A, B = rand_amps(rng, N, n), rand_amps(rng, Nacc, n)
    V = rng.normal(size=(n, 2))
    M = oracle.norm_matrix(B, Nacc + 50)
    f, g, parts = oracle.nll_grad_eq2(A, M, V)
    # (d) definition in numpy: -sum ln|S|^2 + N ln( V^H M V )
    Vc, Ac, Mc = cplx(V), cplx(A), cplx(M)
    norm = (Vc.conj() @ Mc @ Vc).real
    assert f == pytest.approx(-np.log(np.abs(Ac @ Vc) ** 2).sum() + N * math.log(norm), rel=1e-13)
    # (a) scale invariance, and the gradient scales like 1/s
    for s in (0.37, 4.2):
        f2, g2, _ = oracle.nll_grad_eq2(A, M, s * V)
        assert f2 == pytest.approx(f, rel=1e-13)
        assert np.allclose(g2 * s, g, rtol=1e-11, atol=1e-11 * np.abs(g).max())
    assert abs((V * g).sum()) <= 1e-10 * np.abs(g).max()          # Euler: V . grad = 0 (degree-0 homogeneous)
    # (b) central differences
    h = 1e-6
    for a in range(n):
        for c in range(2):
            Vp, Vm = V.copy(), V.copy()
            Vp[a, c] += h
            Vm[a, c] -= h
            fd = (oracle.nll_grad_eq2(A, M, Vp)[0] - oracle.nll_grad_eq2(A, M, Vm)[0]) / (2 * h)
            assert fd == pytest.approx(g[a, c], rel=2e-7, abs=2e-7 * np.abs(g).max())
    # (c) rescale V so that Norm = N: eq. 2 and eq. 3 share the gradient there
    Vs = V * math.sqrt(N / parts[1])
    f3, g3, p3, _ = oracle.nll_grad(A, M, Vs)
    f2, g2, p2 = oracle.nll_grad_eq2(A, M, Vs)
    assert p3[1] == pytest.approx(N, rel=1e-13)
    assert f2 == pytest.approx(f3 - N + N * math.log(N), rel=1e-12)
    assert np.allclose(g2, g3, rtol=1e-10, atol=1e-10 * np.abs(g3).max())


def test_p14_polar_chain_rule(oracle):
    """V_a = r_a exp(i phi_a).  (d/dr, d/dphi) from the Cartesian gradient vs central
    differences taken directly in (r, phi); the sum of d/dphi vanishes (global phase, P2)."""
    rng = np.random.default_rng(14)
    N, Nacc, n = 300, 500, 4
    A, B = rand_amps(rng, N, n), rand_amps(rng, Nacc, n)
    r, phi = rng.uniform(0.3, 2.0, n), rng.uniform(-math.pi, math.pi, n)
    M = oracle.norm_matrix(B, Nacc)

    def f_polar(r, phi):
        V = np.stack([r * np.cos(phi), r * np.sin(phi)], axis=-1)
        return oracle.nll_grad(A, M, V)

    V = np.stack([r * np.cos(phi), r * np.sin(phi)], axis=-1)
    _, g, _, _ = oracle.nll_grad(A, M, V)
    gp = oracle.grad_polar(V, g)
    h = 1e-6
    for a in range(n):
        e = np.zeros(n)
        e[a] = h
        fd_r = (f_polar(r + e, phi)[0] - f_polar(r - e, phi)[0]) / (2 * h)
        fd_p = (f_polar(r, phi + e)[0] - f_polar(r, phi - e)[0]) / (2 * h)
        scale = np.abs(gp).max()
        assert fd_r == pytest.approx(gp[a, 0], rel=2e-7, abs=2e-7 * scale)
        assert fd_p == pytest.approx(gp[a, 1], rel=2e-7, abs=2e-7 * scale)
    assert abs(gp[:, 1].sum()) <= 1e-10 * np.abs(gp).max()


def test_p18_fixed_phase_gauge(oracle):
    """P:85-87 / SURVEY NEXT-4: nll does not depend on a common phase of V; the gauge "wave ref real and >= 0".
    (a) V' keeps every magnitude and every relative phase (V'_a |V_ref| = V_a conj(V_ref), complex arithmetic in numpy),
    Im V'_ref = 0, Re V'_ref = |V_ref|; (b) nll(V') = nll(V) in both likelihood forms; (c) the turned gradient equals the
    gradient the oracle evaluates AT V' (an independent evaluation), except for the dropped component, which is 0;
    (d) gauge identity at any V: sum_a (x_a g_ya - y_a g_xa) = 0 (the derivative along the phase orbit), so the dropped
    component carries no information: g'_y,ref = -sum_{a != ref} (x'_a g'_ya - y'_a g'_xa) / x'_ref; a wrong turning sense
    of the gradient fails (c) and (d)."""
    rng = np.random.default_rng(18)
    N, Nacc, n = 350, 600, 5
    A, B = rand_amps(rng, N, n), rand_amps(rng, Nacc, n)
    M = oracle.norm_matrix(B, Nacc + 20)
    for ref in (0, 3):
        V = rng.normal(size=(n, 2))
        f, g, parts, _ = oracle.nll_grad(A, M, V)
        V2, g2 = oracle.fix_phase(V, g, ref)
        Vc, V2c = cplx(V), cplx(V2)
        assert V2[ref, 1] == 0.0 and V2[ref, 0] == pytest.approx(abs(Vc[ref]), rel=1e-15)
        assert np.allclose(V2c * abs(Vc[ref]), Vc * np.conj(Vc[ref]), rtol=1e-14, atol=1e-15)
        f2, gt, parts2, _ = oracle.nll_grad(A, M, V2)
        assert f2 == pytest.approx(f, rel=1e-13) and parts2[1] == pytest.approx(parts[1], rel=1e-13)
        e2, _, _ = oracle.nll_grad_eq2(A, M, V)
        e2t, _, _ = oracle.nll_grad_eq2(A, M, V2)
        assert e2t == pytest.approx(e2, rel=1e-13)
        scale = np.abs(gt).max()
        mask = np.ones((n, 2), bool)
        mask[ref, 1] = False
        assert np.abs(g2 - gt)[mask].max() <= 1e-11 * scale and g2[ref, 1] == 0.0
        for VV, gg in ((V, g), (V2, gt)):
            assert abs((VV[:, 0] * gg[:, 1] - VV[:, 1] * gg[:, 0]).sum()) <= 1e-10 * scale * np.abs(VV).max()
        others = [a for a in range(n) if a != ref]
        rec = -(V2[others, 0] * gt[others, 1] - V2[others, 1] * gt[others, 0]).sum() / V2[ref, 0]
        assert rec == pytest.approx(gt[ref, 1], rel=1e-8, abs=1e-10 * scale)
        Vonly, none = oracle.fix_phase(V, None, ref)
        assert none is None and np.array_equal(Vonly, V2)


# ---------------------------------------------------------------- P15 Fumili-style approximate Hessian (NEXT-2)
def test_p15_fumili_matrix(oracle):
    """H_data = sum_i u_i u_i^T with u_i = grad ln I_i.  (a) numpy/BLAS restatement; (b) symmetric PSD;
    (c) Euler identity: ln I is homogeneous of degree 0 in V up to ln s^2, so u_i . (x, y) = 2 and
    H_data (x, y) = 2 sum_i u_i = 2 grad(L_data); (d) Hess(Norm) equals the (exact) finite difference of
    the norm gradient 2 M V; (e) u_i itself against central differences of ln I for one event."""
    rng = np.random.default_rng(15)
    N, n = 300, 5
    A, B = rand_amps(rng, N, n), rand_amps(rng, 500, n)
    V = rng.normal(size=(n, 2))
    M = oracle.norm_matrix(B, 520)
    Hd = oracle.fumili(A, V)
    # (a)
    Ac, Vc = cplx(A), cplx(V)
    t = Ac / (Ac @ Vc)[:, None]
    U = np.empty((N, 2 * n))
    U[:, 0::2], U[:, 1::2] = 2 * t.real, -2 * t.imag
    assert np.abs(Hd - U.T @ U).max() <= 1e-12 * np.abs(Hd).max()
    # (b)
    assert np.array_equal(Hd, Hd.T) and np.linalg.eigvalsh(Hd).min() >= -1e-10 * np.trace(Hd)
    # (c)
    L, T, _ = oracle.data_term(A, V)
    gL = np.empty(2 * n)
    gL[0::2], gL[1::2] = 2 * T[:, 0], -2 * T[:, 1]              # grad L_data = 2 conj(T)
    assert np.abs(Hd @ V.reshape(-1) - 2 * gL).max() <= 1e-11 * np.abs(gL).max()
    # (d) Norm is quadratic: central differences of its gradient are exact up to rounding
    H = oracle.fumili(A, V, M)
    HN = H - Hd
    zero = np.zeros((n, 2))
    for p in range(2 * n):
        e = np.zeros(2 * n)
        e[p] = 0.5
        gp = oracle.assemble(0.0, zero, M, (V.reshape(-1) + e).reshape(n, 2))[1].reshape(-1)
        gm = oracle.assemble(0.0, zero, M, (V.reshape(-1) - e).reshape(n, 2))[1].reshape(-1)
        assert np.abs((gp - gm) - HN[:, p]).max() <= 1e-12 * np.abs(HN).max()
    # (e) one event: u = grad ln I by central differences
    H1 = oracle.fumili(A[:1], V)
    h = 1e-6
    u = np.empty(2 * n)
    for p in range(2 * n):
        e = np.zeros(2 * n)
        e[p] = h
        lp = oracle.data_term(A[:1], (V.reshape(-1) + e).reshape(n, 2))[0]
        lm = oracle.data_term(A[:1], (V.reshape(-1) - e).reshape(n, 2))[0]
        u[p] = (lp - lm) / (2 * h)
    assert np.abs(H1 - np.outer(u, u)).max() <= 1e-6 * np.abs(H1).max()


# ---------------------------------------------------------------- P16 per-event weights (NEXT-3)
def test_p16_event_weights(oracle):
    """Weighted sums: (a) w = 1 is bit-identical to the unweighted functions; (b) small integer weights
    = the sample with event i repeated w_i times (exactly the same terms); (c) numpy restatement;
    (d) linearity in w (w1 + w2), incl. negative weights (side-band subtraction style)."""
    rng = np.random.default_rng(16)
    N, n = 600, 4
    A, V = rand_amps(rng, N, n), rng.normal(size=(n, 2))
    one = np.ones(N)
    L0, T0, _ = oracle.data_term(A, V)
    L1, T1, _ = oracle.data_term_w(A, V, one)
    assert L0 == L1 and np.array_equal(T0, T1)
    assert np.array_equal(oracle.norm_matrix(A, N + 3), oracle.norm_matrix_w(A, N + 3, one))
    k = rng.integers(0, 4, size=N)
    Arep = np.repeat(A, k, axis=0)
    Lw, Tw, _ = oracle.data_term_w(A, V, k.astype(float))
    Lr, Tr, _ = oracle.data_term(Arep, V)
    assert Lw == pytest.approx(Lr, rel=1e-13) and np.allclose(Tw, Tr, rtol=1e-12, atol=1e-12 * np.abs(Tr).max())
    Mw, Mr = oracle.norm_matrix_w(A, 777, k.astype(float)), oracle.norm_matrix(Arep, 777)
    assert np.abs(Mw - Mr).max() <= 1e-13 * np.abs(Mr).max()
    w = rng.normal(size=N)
    Ac, Vc = cplx(A), cplx(V)
    S = Ac @ Vc
    Lw, Tw, _ = oracle.data_term_w(A, V, w)
    assert Lw == pytest.approx((w * np.log(np.abs(S) ** 2)).sum(), rel=1e-12)
    assert np.abs(cplx(Tw) - (w[:, None] * Ac / S[:, None]).sum(0)).max() <= 1e-12 * np.abs(Tw).max()
    Mw = cplx(oracle.norm_matrix_w(A, 900, w))
    assert np.abs(Mw - (Ac.conj().T * w) @ Ac / 900).max() <= 1e-13 * np.abs(Mw).max()
    w2 = rng.normal(size=N)
    La, Ta, _ = oracle.data_term_w(A, V, w2)
    Lb, Tb, _ = oracle.data_term_w(A, V, w + w2)
    assert Lb == pytest.approx(Lw + La, rel=1e-11, abs=1e-11 * (abs(Lw) + abs(La)))
    assert np.allclose(Tb, Tw + Ta, rtol=1e-11, atol=1e-11 * np.abs(Tb).max())


# ---------------------------------------------------------------- P17 sampled-block entry points (offset indexing)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_p17_norm_block_offsets(oracle, dtype):
    """norm_block(a0, a1, b0, b1) with a0, b0 > 0 (the indexing every full-size M check rests on):
    the block equals the same entries of the full matrix BITWISE (same per-event terms, same order),
    entries outside the block stay 0, and the block equals the numpy/BLAS restatement
    M_ab = (1/N_gen) sum_j conj(B_ja) B_jb (P:41 inner bracket, C1) — non-square blocks with a != b
    ranges so a transposed or shifted index fails."""
    rng = np.random.default_rng(17)
    n, Nacc, Ngen = 7, 1501, 1777
    B = rand_amps(rng, Nacc, n).astype(dtype)
    w = rng.uniform(0.2, 2.0, size=Nacc)
    full = oracle.norm_matrix(B, Ngen)
    full_w = oracle.norm_matrix_w(B, Ngen, w)
    Bc = cplx(B.astype(np.float64))
    M_np = Bc.conj().T @ Bc / Ngen
    M_np_w = (Bc.conj().T * w) @ Bc / Ngen
    assert np.abs(cplx(full) - M_np).max() <= 1e-13 * np.abs(M_np).max()
    for a0, a1, b0, b1 in [(2, 5, 1, 7), (3, 4, 6, 7), (6, 7, 0, 2), (1, 7, 3, 5), (0, 7, 0, 7), (4, 4, 2, 6)]:
        blk = oracle.norm_block(B, Ngen, a0, a1, b0, b1)
        assert np.array_equal(blk[a0:a1, b0:b1], full[a0:a1, b0:b1]), (a0, a1, b0, b1)
        outside = blk.copy()
        outside[a0:a1, b0:b1] = 0.0
        assert not outside.any()
        if a1 > a0:
            assert np.abs(cplx(blk)[a0:a1, b0:b1] - M_np[a0:a1, b0:b1]).max() <= 1e-13 * np.abs(M_np).max()
        # the weighted entry point with offsets (called directly: the Python wrapper only passes 0..n)
        blk_w = np.zeros((n, n, 2))
        Bx, dt = oracle._amp(B)
        oracle.lib().pwa_oracle_norm_block_w(oracle._p(Bx), dt, oracle.C.c_int64(Nacc), n, oracle.C.c_int64(Ngen),
                                             oracle._p(w), a0, a1, b0, b1, oracle._p(blk_w))
        assert np.array_equal(blk_w[a0:a1, b0:b1], full_w[a0:a1, b0:b1])
        if a1 > a0:
            assert np.abs(cplx(blk_w)[a0:a1, b0:b1] - M_np_w[a0:a1, b0:b1]).max() <= 1e-13 * np.abs(M_np_w).max()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_p17_fumili_rows_offsets(oracle, dtype):
    """fumili_rows(p0, p1) with p0 > 0: rows equal the full matrix bitwise, other rows stay 0, and
    the rows equal the numpy restatement sum_i u_i[p] u_i[q]."""
    rng = np.random.default_rng(18)
    N, n = 401, 5
    A = rand_amps(rng, N, n).astype(dtype)
    V = rng.normal(size=(n, 2))
    full = oracle.fumili(A, V)
    Ac, Vc = cplx(A.astype(np.float64)), cplx(V)
    t = Ac / (Ac @ Vc)[:, None]
    U = np.empty((N, 2 * n))
    U[:, 0::2], U[:, 1::2] = 2 * t.real, -2 * t.imag
    H_np = U.T @ U
    for p0, p1 in [(1, 3), (4, 5), (9, 10), (3, 10), (0, 10)]:
        rows = oracle.fumili_rows(A, V, p0, p1)
        assert np.array_equal(rows[p0:p1], full[p0:p1]), (p0, p1)
        assert not rows[:p0].any() and not rows[p1:].any()
        assert np.abs(rows[p0:p1] - H_np[p0:p1]).max() <= 1e-12 * np.abs(H_np).max()
