"""Pins for the oracle's DM steps (oracle/dm_oracle.c), chosen so that a dropped term, a
wrong sign, index or conjugate, or a transposed operand fails at least one of them.

Expected values come from: closed forms of eqs. (3)-(7), invariants,
special cases that reduce to textbook operations, and an independent numpy restatement
with dense DFT matrices on a tiny case.  None of them comes from the CUDA path.
"""
import numpy as np
import pytest

import oracle
from paper_1808_10375_b200 import synth


# ----------------------------------------------------------------- helpers ----
def dft_matrix(n):
    k = np.arange(n)
    return np.exp(-2j * np.pi * np.outer(k, k) / n)


def windows(O, pos, n):
    """O [L][H][W], pos [J][2] -> [J][L][n][n]."""
    return np.stack([np.stack([O[l, y:y + n, x:x + n] for l in range(O.shape[0])]) for y, x in pos])


def numpy_dm_iteration(P, O, psi, amp, pos, beta, alpha_o, alpha_p, eps=1e-30):
    """Independent restatement of one DM iteration (order A3/A4) with dense DFT matrices.
    psi [J][K][L][n][n].  Returns P_new, O_new, psi_new, error row."""
    J, K, L, n, _ = psi.shape
    Fm = dft_matrix(n)
    Fi = np.conj(Fm) / n
    win = windows(O, pos, n)                                     # [J][L][n][n]
    PO = P[None, :, None] * win[:, None]                          # [J][K][L][n][n]
    R = 2 * PO - psi
    F = np.einsum("vy,jklyx,ux->jklvu", Fm, R, Fm)
    S = (np.abs(F) ** 2).sum(axis=(1, 2))                         # [J][n][n]
    scale = amp / np.sqrt(S + eps)
    G = np.einsum("yv,jklvu,xu->jklyx", Fi, F * scale[:, None, None], Fi)
    d = beta * (G - PO)
    psi_new = psi + d
    eF = np.sqrt(((np.sqrt(S) - amp) ** 2).sum() / (amp ** 2).sum())
    epsi = np.sqrt((np.abs(d) ** 2).sum() / (np.abs(psi_new) ** 2).sum())
    # object, eq. (6): old P, new psi
    num = np.zeros_like(O)
    den = np.zeros(O.shape[1:])
    for j, (y, x) in enumerate(pos):
        for k in range(K):
            den[y:y + n, x:x + n] += np.abs(P[k]) ** 2
            for l in range(L):
                num[l, y:y + n, x:x + n] += np.conj(P[k]) * psi_new[j, k, l]
    tot = alpha_o + den
    O_new = np.where(tot > 0, (alpha_o * O + num) / np.where(tot > 0, tot, 1), O)
    # probe, eq. (5): new O, new psi
    win = windows(O_new, pos, n)
    nump = np.einsum("jlyx,jklyx->kyx", np.conj(win), psi_new)
    denp = (np.abs(win) ** 2).sum(axis=(0, 1))
    P_new = (alpha_p * P + nump) / (alpha_p + denp)
    eP = [np.sqrt((np.abs(P_new[k] - P[k]) ** 2).sum() / (np.abs(P_new[k]) ** 2).sum()) for k in range(K)]
    eO = [np.sqrt((np.abs(O_new[l] - O[l]) ** 2).sum() / (np.abs(O_new[l]) ** 2).sum()) for l in range(L)]
    return P_new, O_new, psi_new, np.array([eF, epsi] + eP + eO)


def tiny_problem(rng, n=8, K=2, L=1, H=14, W=16, pos=((0, 0), (1, 5), (5, 2), (6, 8))):
    pos = np.array(pos, np.int32)
    P = (rng.standard_normal((K, n, n)) + 1j * rng.standard_normal((K, n, n))).astype(np.complex64)
    O = (1 + 0.3 * rng.standard_normal((L, H, W)) + 0.3j * rng.standard_normal((L, H, W))).astype(np.complex64)
    win = windows(O.astype(complex), pos, n)
    psi_true = P.astype(complex)[None, :, None] * win[:, None]
    I = (np.abs(np.fft.fft2(psi_true)) ** 2).sum(axis=(1, 2))       # float64: exactly consistent
    return pos, P, O, I


# ------------------------------------------------ modulus projection, eq. (4) ----
def test_modulus_projection_textbook_single_mode(rng):
    n = 16
    F = rng.standard_normal((1, n, n)) + 1j * rng.standard_normal((1, n, n))
    amp = rng.uniform(0.1, 2.0, (n, n))
    out, err = oracle.modulus_project(F, amp, eps=0.0)
    want = amp * np.exp(1j * np.angle(F[0]))                      # replace modulus, keep phase
    assert np.abs(out[0] - want).max() < 1e-13
    assert abs(err - ((np.abs(F[0]) - amp) ** 2).sum()) < 1e-10


def test_modulus_projection_mode_sum_and_idempotence(rng):
    n, M = 16, 3
    F = rng.standard_normal((M, n, n)) + 1j * rng.standard_normal((M, n, n))
    amp = rng.uniform(0.1, 2.0, (n, n))
    out, _ = oracle.modulus_project(F, amp)
    assert np.abs((np.abs(out) ** 2).sum(0) - amp ** 2).max() < 1e-12     # eq. (1) holds after F_c
    # the ratio between modes is kept (common real scale), phases kept
    assert np.abs(out[1] * F[0] - out[0] * F[1]).max() < 1e-12
    assert np.abs(np.angle(out * np.conj(F))).max() < 1e-12
    out2, err2 = oracle.modulus_project(out, amp)
    assert np.abs(out2 - out).max() < 1e-12                                # idempotent
    assert err2 < 1e-20


def test_modulus_projection_zero_spectrum_is_guarded():
    n = 8
    F = np.zeros((2, n, n), complex)
    out, err = oracle.modulus_project(F, np.ones((n, n)))
    assert np.all(out == 0) and np.isfinite(err) and abs(err - n * n) < 1e-12


# ------------------------------------------------------- psi update, eq. (3) ----
@pytest.mark.parametrize("beta", [1.0, 0.8, 0.3])
def test_psi_update_fixed_point_on_consistent_data(rng, beta):
    pos, P, O, I = tiny_problem(rng, K=2, L=2)
    amp = np.sqrt(I.astype(float))
    for j, (y, x) in enumerate(pos):
        psi = P.astype(complex)[:, None] * O.astype(complex)[None, :, y:y + 8, x:x + 8]
        new, acc = oracle.view_update(P, O, y, x, psi, amp[j], beta=beta)
        assert np.abs(new - psi).max() < 1e-10
        assert acc[0] < 1e-20 * acc[1] and acc[2] < 1e-20 * acc[3]


def test_psi_update_beta_zero_keeps_psi(rng):
    pos, P, O, I = tiny_problem(rng)
    psi = rng.standard_normal((2, 1, 8, 8)) + 1j * rng.standard_normal((2, 1, 8, 8))
    new, _ = oracle.view_update(P, O, 1, 5, psi, np.sqrt(I[1].astype(float)), beta=0.0)
    assert np.abs(new - psi).max() < 1e-14


def test_psi_update_first_step_is_error_reduction(rng):
    # psi = PO and beta = 1  =>  psi_new = IFFT[ sqrt(I)/sqrt(S) FFT(PO) ]  (plain projection)
    pos, P, O, _ = tiny_problem(rng)
    amp = rng.uniform(0.5, 3.0, (8, 8))
    y, x = pos[2]
    PO = P.astype(complex)[:, None] * O.astype(complex)[None, :, y:y + 8, x:x + 8]
    F = np.fft.fft2(PO)
    want = np.fft.ifft2(F * amp / np.sqrt((np.abs(F) ** 2).sum((0, 1))))
    new, acc = oracle.view_update(P, O, y, x, PO, amp, beta=1.0)
    assert np.abs(new - want).max() < 1e-12
    S = (np.abs(F) ** 2).sum((0, 1))
    assert abs(acc[0] - ((np.sqrt(S) - amp) ** 2).sum()) < 1e-9 * acc[0]
    assert abs(acc[1] - (amp ** 2).sum()) < 1e-12 * acc[1]
    assert abs(acc[2] - (np.abs(want - PO) ** 2).sum()) < 1e-9 * acc[2]
    assert abs(acc[3] - (np.abs(want) ** 2).sum()) < 1e-12 * acc[3]


@pytest.mark.parametrize("beta", [1.0, 0.8])
def test_psi_update_fused_form_identity(rng, beta):
    # psi + beta(IFFT[scale F] - PO) == (2-beta) PO + IFFT[(beta scale - 1) F]
    pos, P, O, I = tiny_problem(rng, K=2, L=2)
    psi = rng.standard_normal((2, 2, 8, 8)) + 1j * rng.standard_normal((2, 2, 8, 8))
    amp = np.sqrt(I[0].astype(float))
    a, acc_a = oracle.view_update(P, O, 0, 0, psi, amp, beta=beta, fused=False)
    b, acc_b = oracle.view_update(P, O, 0, 0, psi, amp, beta=beta, fused=True)
    assert np.abs(a - b).max() < 1e-12
    assert np.allclose(acc_a, acc_b, rtol=1e-10)


# ----------------------------------------- overlap projection, eqs. (5), (6) ----
def test_object_update_returns_object_on_consistent_psi(rng):
    pos, P, O, _ = tiny_problem(rng, K=2, L=2)
    Oc, Pc = O.astype(complex), P.astype(complex)
    psi = Pc[None, :, None] * windows(Oc, pos, 8)[:, None]
    cov = oracle.cover_count(8, pos, *O.shape[1:]) > 0
    for alpha in (0.0, 0.7):
        O_old = Oc if alpha else np.full_like(Oc, 9 - 3j)   # alpha=0: old value must not leak in
        got = oracle.object_update(pos, P, psi, O_old, alpha=alpha)
        assert np.abs(got[:, cov] - Oc[:, cov]).max() < 1e-12
        assert np.abs(got[:, ~cov] - O_old[:, ~cov]).max() < 1e-15      # uncovered: keep old


def test_probe_update_returns_probe_on_consistent_psi(rng):
    pos, P, O, _ = tiny_problem(rng, K=2, L=2)
    Oc, Pc = O.astype(complex), P.astype(complex)
    psi = Pc[None, :, None] * windows(Oc, pos, 8)[:, None]
    got = oracle.probe_update(pos, O, psi, np.full_like(Pc, 5 + 1j), alpha=0.0)
    assert np.abs(got - Pc).max() < 1e-12
    got = oracle.probe_update(pos, O, psi, Pc, alpha=0.3)
    assert np.abs(got - Pc).max() < 1e-12


def test_single_view_object_update_is_pointwise_quotient(rng):
    n = 8
    P = rng.standard_normal((1, n, n)) + 1j * rng.standard_normal((1, n, n))
    psi = rng.standard_normal((1, 1, 1, n, n)) + 1j * rng.standard_normal((1, 1, 1, n, n))
    O_old = np.zeros((1, 12, 12), complex)
    got = oracle.object_update([(2, 3)], P, psi, O_old)
    assert np.abs(got[0, 2:10, 3:11] - psi[0, 0, 0] / P[0]).max() < 1e-12


def test_overlap_updates_against_numpy_scatter_restatement(rng):
    pos, P, O, _ = tiny_problem(rng, K=2, L=2)
    J, n = len(pos), 8
    psi = rng.standard_normal((J, 2, 2, n, n)) + 1j * rng.standard_normal((J, 2, 2, n, n))
    Pc, Oc = P.astype(complex), O.astype(complex)
    num = np.zeros_like(Oc)
    den = np.zeros(Oc.shape[1:])
    for j, (y, x) in enumerate(pos):
        for k in range(2):
            den[y:y + n, x:x + n] += np.abs(Pc[k]) ** 2
            for l in range(2):
                num[l, y:y + n, x:x + n] += np.conj(Pc[k]) * psi[j, k, l]
    alpha = 0.25
    want = (alpha * Oc + num) / (alpha + den)
    assert np.abs(oracle.object_update(pos, P, psi, O, alpha=alpha) - want).max() < 1e-12
    win = windows(Oc, pos, n)
    nump = np.einsum("jlyx,jklyx->kyx", np.conj(win), psi)
    denp = (np.abs(win) ** 2).sum((0, 1))
    wantp = (alpha * Pc + nump) / (alpha + denp)
    assert np.abs(oracle.probe_update(pos, O, psi, P, alpha=alpha) - wantp).max() < 1e-12


def test_object_update_minimises_least_squares(rng):
    # eq. (6) with alpha = 0 is the minimiser over O of sum |psi - P O|^2 for fixed P
    pos, P, O, _ = tiny_problem(rng, K=2, L=1)
    J, n = len(pos), 8
    psi = rng.standard_normal((J, 2, 1, n, n)) + 1j * rng.standard_normal((J, 2, 1, n, n))
    Pc = P.astype(complex)

    def cost(Ox):
        return sum((np.abs(psi[j, k, 0] - Pc[k] * Ox[0, y:y + n, x:x + n]) ** 2).sum()
                   for j, (y, x) in enumerate(pos) for k in range(2))

    best = oracle.object_update(pos, P, psi, O.astype(complex), alpha=0.0)
    c0 = cost(best)
    for _ in range(20):
        d = 1e-3 * (rng.standard_normal(best.shape) + 1j * rng.standard_normal(best.shape))
        assert cost(best + d) > c0
    # and likewise eq. (5) over P for fixed O
    def costp(Px):
        return sum((np.abs(psi[j, k, 0] - Px[k] * best[0, y:y + n, x:x + n]) ** 2).sum()
                   for j, (y, x) in enumerate(pos) for k in range(2))
    pbest = oracle.probe_update(pos, best, psi, Pc, alpha=0.0)
    c1 = costp(pbest)
    for _ in range(20):
        d = 1e-3 * (rng.standard_normal(pbest.shape) + 1j * rng.standard_normal(pbest.shape))
        assert costp(pbest + d) > c1


# ------------------------------------------------------------ error metric ----
def test_rel_change_closed_forms(rng):
    a = rng.standard_normal(50) + 1j * rng.standard_normal(50)
    assert oracle.rel_change(a, a) == 0.0
    assert abs(oracle.rel_change(a, np.zeros_like(a)) - 1.0) < 1e-15
    assert oracle.rel_change(np.zeros_like(a), np.zeros_like(a)) == 0.0
    assert abs(oracle.rel_change(2 * a, a) - 0.5) < 1e-15          # eq. (7): normalised by NEW


# ------------------------------------------------------- whole iterations ----
@pytest.mark.parametrize("K,L,beta,a", [(2, 1, 1.0, 1e-3), (2, 2, 0.8, 0.0), (1, 1, 1.0, 0.0), (3, 2, 0.5, 1e-2)])
def test_three_iterations_against_dense_dft_restatement(rng, K, L, beta, a):
    pos, P, O, I = tiny_problem(rng, K=K, L=L)
    I = (I * rng.uniform(0.7, 1.3, I.shape)).astype(np.float32)          # make it inconsistent; float32 as the ABI takes
    P0 = (0.9 * P).astype(np.complex64)
    O0 = np.ones_like(O)
    if L > 1:
        O0[1:] = (0.1 * (rng.standard_normal(O0[1:].shape) + 1j * rng.standard_normal(O0[1:].shape)))
    o = oracle.OracleDM(8, K, L, O.shape[1], O.shape[2], pos, beta=beta, alpha_obj=a, alpha_probe=a)
    o.set_data(I, P0, O0)
    Pn, On = P0.astype(complex), O0.astype(complex)
    psi = Pn[None, :, None] * windows(On, pos, 8)[:, None]
    assert np.abs(o.psi() - psi).max() < 1e-14
    # frozen regularisers (reading A8)
    den = np.zeros(O.shape[1:])
    for y, x in pos:
        den[y:y + 8, x:x + 8] += (np.abs(Pn) ** 2).sum(0)
    a_o = a * den.max()
    a_p = a * (np.abs(windows(On, pos, 8)) ** 2).sum((0, 1)).max()
    assert np.allclose(o.alphas, (a_o, a_p), rtol=1e-13, atol=0)
    amp = np.sqrt(I.astype(float))
    rows = []
    for _ in range(3):
        Pn, On, psi, row = numpy_dm_iteration(Pn, On, psi, amp, pos, beta, a_o, a_p)
        rows.append(row)
    o.iterate(3)
    assert np.abs(o.psi() - psi).max() < 1e-10
    assert np.abs(o.probe() - Pn).max() < 1e-10
    assert np.abs(o.object() - On).max() < 1e-10
    assert np.abs(o.errors() - np.array(rows)).max() < 1e-10


def test_noise_free_truth_is_a_fixed_point_of_the_whole_iteration():
    pr = synth.make_problem(synth.CONFIGS[0].scaled(3, 3))
    c = pr.cfg
    # exact data for the complex64 truth, so that psi = P O is consistent to rounding
    Pt, Ot = pr.probe_true.astype(complex), pr.object_true.astype(complex)
    psi = Pt[None, :, None] * windows(Ot, pr.positions, c.N)[:, None]
    I = (np.abs(np.fft.fft2(psi)) ** 2).sum((1, 2))
    o = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions)
    o.set_data(I.astype(np.float32), pr.probe_true, pr.object_true)
    o.iterate(1)
    cov = oracle.cover_count(c.N, pr.positions, c.obj_h, c.obj_w) > 0
    # float32 storage of I limits consistency to ~1e-7 relative
    assert synth.rel_l2(o.psi(), psi) < 1e-6
    assert synth.rel_l2(o.probe(), Pt) < 1e-6
    assert np.abs(o.object()[:, cov] - Ot[:, cov]).max() < 1e-4
    assert np.all(o.errors()[0] < 1e-6)


# ------------------------------------------------------------ equivariances ----
def _run(pr, n_it=2, **kw):
    c = pr.cfg
    o = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions, **kw)
    o.set_data(pr.intensities, pr.probe0, pr.object0)
    o.iterate(n_it)
    return o


def test_equivariance_global_phase_and_scale_exchange():
    pr = synth.make_problem(synth.CONFIGS[1].scaled(3, 3))
    base = _run(pr)
    # exact factors (i, 2, 1/2) so both runs start from representable numbers: a rounded
    # start differs by ~1e-7 and DM amplifies that (A20/A21)
    ph = np.complex64(1j)
    pr2 = synth.DMProblem(**{**pr.__dict__, "probe0": (pr.probe0 * ph).astype(np.complex64)})
    rot = _run(pr2)
    assert synth.rel_l2(rot.probe(), base.probe() * complex(ph)) < 1e-12
    assert synth.rel_l2(rot.object(), base.object()) < 1e-12
    assert np.abs(rot.errors() - base.errors()).max() < 1e-12
    pr3 = synth.DMProblem(**{**pr.__dict__, "probe0": pr.probe0 * np.float32(2.0),
                             "object0": pr.object0 * np.float32(0.5)})
    ex = _run(pr3)
    assert synth.rel_l2(ex.psi(), base.psi()) < 1e-12
    assert synth.rel_l2(ex.probe(), 2 * base.probe()) < 1e-12


def test_equivariance_translation_and_view_permutation():
    pr = synth.make_problem(synth.CONFIGS[0].scaled(3, 4))
    c = pr.cfg
    base = _run(pr, alpha_obj=0.0, alpha_probe=0.0)
    dy, dx = 5, 8
    big = np.ones((c.L, c.obj_h + dy + 3, c.obj_w + dx + 2), np.complex64)
    big[:, dy:dy + c.obj_h, dx:dx + c.obj_w] = pr.object0
    o = oracle.OracleDM(c.N, c.K, c.L, big.shape[1], big.shape[2], pr.positions + np.array([dy, dx], np.int32),
                        alpha_obj=0.0, alpha_probe=0.0)
    o.set_data(pr.intensities, pr.probe0, big)
    o.iterate(2)
    assert np.abs(o.probe() - base.probe()).max() == 0.0
    assert np.abs(o.object()[:, dy:dy + c.obj_h, dx:dx + c.obj_w] - base.object()).max() == 0.0
    perm = np.random.default_rng(5).permutation(c.n_views)
    pr_p = synth.DMProblem(**{**pr.__dict__, "positions": pr.positions[perm], "intensities": pr.intensities[perm]})
    p = _run(pr_p, alpha_obj=0.0, alpha_probe=0.0)
    assert synth.rel_l2(p.probe(), base.probe()) < 1e-12
    assert synth.rel_l2(p.object(), base.object()) < 1e-12
    assert synth.rel_l2(p.psi(), base.psi()[perm]) < 1e-12


def test_set_state_round_trip_and_teacher_forcing():
    pr = synth.make_problem(synth.CONFIGS[0].scaled(3, 3))
    a = _run(pr, n_it=3)
    b = _run(pr, n_it=1)
    c = pr.cfg
    fresh = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions)
    fresh.set_data(pr.intensities, pr.probe0, pr.object0)
    fresh.set_state(b.probe(), b.object(), b.psi())
    fresh.iterate(2)
    assert np.abs(fresh.probe() - a.probe()).max() == 0.0
    assert np.abs(fresh.psi() - a.psi()).max() == 0.0


def test_create_rejects_bad_arguments():
    with pytest.raises(ValueError):
        oracle.OracleDM(8, 1, 1, 10, 10, [(3, 0)])          # window leaves the object
    with pytest.raises(ValueError):
        oracle.OracleDM(12, 1, 1, 20, 20, [(0, 0)])         # not a power of two
    o = oracle.OracleDM(8, 1, 1, 10, 10, [(0, 0)])
    with pytest.raises(ValueError):
        o.set_param("beta", 1.5)
    with pytest.raises(RuntimeError):
        o.iterate(1)                                         # no data yet


def test_mode_power_closed_form():
    """Mode diagnostics: the synthetic probe modes are sqrt(w_k) * roll(base), so their
    power fractions are the weights w_k exactly; a mode scaled by c changes its share by c^2."""
    for ci in (1, 2, 3, 4):
        cfg = synth.CONFIGS[ci]
        P = synth.make_probe(cfg)
        f = oracle.mode_power(P)
        assert np.allclose(f, np.array(cfg.weights) / sum(cfg.weights), rtol=0, atol=1e-12)
        assert abs(f.sum() - 1.0) < 1e-14
    x = np.ones((2, 4, 4), np.complex128)
    x[1] *= 3j
    assert np.allclose(oracle.mode_power(x), [0.1, 0.9])
    assert np.all(oracle.mode_power(np.zeros((3, 2, 2))) == 0.0)


# ------------------------------------------- view-range entry points (streaming) ----
# Justification of these oracle entry points: eqs. (5), (6) are sums over the views; carried in an
# accumulator over consecutive view ranges they perform the additions of the monolithic functions in their order
# (readings A3, A15).  Pin: bit-identical to oracle_object_update / oracle_probe_update / OracleDM for any split.
@pytest.mark.parametrize("K,L", [(2, 1), (2, 2), (1, 3)])
def test_range_accumulators_are_bit_identical_to_the_monolithic_updates(rng, K, L):
    pos = np.array([(0, 0), (1, 5), (5, 2), (6, 8), (3, 3), (0, 7), (6, 0)], np.int32)
    n, H, W = 8, 15, 16
    P = rng.normal(size=(K, n, n)) + 1j * rng.normal(size=(K, n, n))
    O = rng.normal(size=(L, H, W)) + 1j * rng.normal(size=(L, H, W))
    psi = rng.normal(size=(len(pos), K, L, n, n)) + 1j * rng.normal(size=(len(pos), K, L, n, n))
    for alpha in (0.0, 0.37):
        O_ref = oracle.object_update(pos, P, psi, O, alpha)
        P_ref = oracle.probe_update(pos, O_ref, psi, P, alpha)
        for cuts in ([0, 7], [0, 1, 7], [0, 3, 4, 7], [0, 2, 2, 5, 7], list(range(8))):      # incl. an empty range
            numO, denO = np.zeros((L, H, W), np.complex128), np.zeros((H, W))
            numP, denP = np.zeros((K, n, n), np.complex128), np.zeros((n, n))
            for j0, j1 in zip(cuts[:-1], cuts[1:]):
                oracle.object_accumulate(pos, j0, j1, P, psi[j0:j1], numO, denO)
            O_new = oracle.object_finish(numO, denO, O, alpha)
            assert np.array_equal(O_new, O_ref), (alpha, cuts)
            for j0, j1 in zip(cuts[:-1], cuts[1:]):
                oracle.probe_accumulate(pos, j0, j1, O_new, psi[j0:j1], numP, denP)
            assert np.array_equal(oracle.probe_finish(numP, denP, P, alpha), P_ref), (alpha, cuts)
    # uncovered object pixels keep the old value under the literal quotient (row 14 is outside every window)
    assert np.array_equal(oracle.object_update(pos, P, psi, O, 0.0)[:, 14], O[:, 14])


def test_views_update_and_frozen_alphas_match_the_stateful_oracle():
    pr = synth.make_problem(synth.CONFIGS[1].scaled(3, 4))
    c = pr.cfg
    o = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions, beta=0.8)
    o.set_data(pr.intensities, pr.probe0, pr.object0)
    assert oracle.frozen_alphas(pr.positions, pr.probe0, pr.object0) == o.alphas
    P, O, psi0 = o.probe(), o.object(), o.psi()
    amp = np.sqrt(pr.intensities.astype(np.float64))
    got, acc = oracle.views_update(pr.positions, 2, 9, P, O, psi0[2:9], amp[2:9], beta=0.8)
    for j in range(2, 9):
        y0, x0 = pr.positions[j]
        want, a = oracle.view_update(P, O, y0, x0, psi0[j], amp[j], beta=0.8)
        assert np.array_equal(got[j - 2], want) and np.array_equal(acc[j - 2], a)
    o.close()


class _DictStash:
    def __init__(self):
        self.d = {}

    def put(self, j0, j1, x):
        self.d[(j0, j1)] = x.copy()

    def get(self, j0, j1):
        return self.d[(j0, j1)]


@pytest.mark.parametrize("cfg_i,ny,nx,chunk,use_stash", [(1, 3, 4, 5, False), (3, 2, 2, 1, True), (0, 4, 4, 16, False),
                                                         (1, 3, 4, 100, True), (1, 3, 4, 5, True)])
def test_streamed_iteration_is_bit_identical_to_oracle_iterate(cfg_i, ny, nx, chunk, use_stash):
    """tests/streamed_oracle.py (what the full-size GPU parity tests of configs 3 and 4 use) against OracleDM.iterate:
    two iterations, the second from the state of the first, psi, P, O and the error rows bit for bit."""
    import streamed_oracle
    pr = synth.make_problem(synth.CONFIGS[cfg_i].scaled(ny, nx))
    c = pr.cfg
    o = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions)
    o.set_data(pr.intensities, pr.probe0, pr.object0)
    a_o, a_p = oracle.frozen_alphas(pr.positions, pr.probe0, pr.object0)
    amp = np.sqrt(pr.intensities.astype(np.float64))
    P, O, psi = o.probe(), o.object(), o.psi()
    for it in range(2):
        new_psi = np.empty_like(psi)

        def keep(j0, j1, chunk_psi):
            new_psi[j0:j1] = chunk_psi
        P, O, row = streamed_oracle.iteration(pr.positions, P, O, lambda a, b: psi[a:b], lambda a, b: amp[a:b],
                                              a_o, a_p, chunk=chunk, on_psi=keep,
                                              stash=_DictStash() if use_stash else None)
        psi = new_psi
        o.iterate(1)
        assert np.array_equal(P, o.probe()) and np.array_equal(O, o.object()) and np.array_equal(psi, o.psi())
        assert np.array_equal(row, o.errors()[it]), (row, o.errors()[it])
    o.close()
