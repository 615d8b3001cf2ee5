"""Pins for the CPU oracle (oracle/rgf_oracle.c): everything here runs without a GPU.

Each test ties the oracle to something other than itself: a closed form, the plain
definition evaluated with LAPACK (numpy) on a matrix this file assembles on its own, an
invariant of the physics, or a statement the paper prints.  No expected value here comes
from the CUDA path.
"""
import os

import numpy as np
import pytest

from paper_1107_5300_b200 import inputs

T_HOP = -2.7
ETA = 1e-9
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------------------
# Independent helpers (written here, not shared with the oracle or the CUDA path)
# ----------------------------------------------------------------------------------------

def closed_form_T(M, L, E, t=T_HOP, eta=ETA):
    """Clean armchair ribbon: T = sum over open subbands of exp(-2 eta L / v_p).

    Transverse modes sin(p pi (j+1)/(M+1)) reduce the ribbon to dimer chains with hoppings
    2 t c_p (inside a slice) and t (between slices), c_p = cos(p pi/(M+1)), p = 1..M//2:
        E^2 = t^2 (1 + 4 c_p^2 + 4 c_p cos k),  k = phase per slice,
    open iff |1 - 2 c_p| < |E/t| < 1 + 2 c_p; group velocity v_p = |dE/dk| = 2 t^2 c_p |sin k| / |E|.
    A uniform i*eta damps each channel by exp(-2 eta L / v_p).
    Returns (T, n_open, distance to the nearest subband edge in eV).
    """
    x = abs(E / t)
    T, n_open, dmin = 0.0, 0, np.inf
    for p in range(1, M // 2 + 1):
        c = np.cos(p * np.pi / (M + 1))
        lo, hi = abs(1 - 2 * c), 1 + 2 * c
        dmin = min(dmin, abs(x - lo) * abs(t), abs(x - hi) * abs(t))
        if lo < x < hi:
            cosk = (x * x - 1 - 4 * c * c) / (4 * c)
            sink = np.sqrt(max(0.0, 1 - cosk * cosk))
            v = 2 * t * t * c * sink / abs(E)
            T += np.exp(-2 * eta * L / v)
            n_open += 1
    return T, n_open, dmin


def mask(i, M):
    return np.array([1.0 if ((i + j) % 2 == 0) else 0.0 for j in range(M)])


def slice_H(M, onsite_row, t, vac_row=None):
    H = np.diag(np.asarray(onsite_row, dtype=float)).astype(complex)
    for j in range(M - 1):
        if vac_row is None or (not vac_row[j] and not vac_row[j + 1]):
            H[j, j + 1] = H[j + 1, j] = t
    return H


def definition_T(onsite, vac, t, E, eta, gL, gR, delete_vacant=False):
    """Eq. 1 + Eq. 2 written out with numpy: invert the whole device, take block (L-1, 0).

    gL, gR: lead surface Green's functions (slices -1 and L).  If delete_vacant, vacant sites
    are REMOVED from the matrix instead of being kept as isolated levels (Q15 pin).
    """
    L, M = onsite.shape
    N = M * L
    H = np.zeros((N, N), dtype=complex)
    isvac = np.zeros((L, M), dtype=bool) if vac is None else vac.astype(bool)
    for i in range(L):
        H[i * M:(i + 1) * M, i * M:(i + 1) * M] = slice_H(M, onsite[i], t, isvac[i])
        if i + 1 < L:
            m = mask(i, M) * (~isvac[i]) * (~isvac[i + 1])
            H[i * M:(i + 1) * M, (i + 1) * M:(i + 2) * M] = np.diag(t * m)
            H[(i + 1) * M:(i + 2) * M, i * M:(i + 1) * M] = np.diag(t * m)
    mL = mask(-1, M) * (~isvac[0])
    mR = mask(L - 1, M) * (~isvac[L - 1])
    SigL = (t * mL)[:, None] * gL * (t * mL)[None, :]
    SigR = (t * mR)[:, None] * gR * (t * mR)[None, :]
    S = np.zeros((N, N), dtype=complex)
    S[:M, :M] += SigL
    S[N - M:, N - M:] += SigR
    A = (E + 1j * eta) * np.eye(N) - H - S
    GamL = np.zeros((N, N), dtype=complex)
    GamR = np.zeros((N, N), dtype=complex)
    GamL[:M, :M] = 1j * (SigL - SigL.conj().T)
    GamR[N - M:, N - M:] = 1j * (SigR - SigR.conj().T)
    if delete_vacant:
        keep = ~isvac.reshape(-1)
        A, GamL, GamR = A[np.ix_(keep, keep)], GamL[np.ix_(keep, keep)], GamR[np.ix_(keep, keep)]
    G = np.linalg.inv(A)
    return np.trace(GamL @ G.conj().T @ GamR @ G).real


# ----------------------------------------------------------------------------------------
# Dense helpers against LAPACK
# ----------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [1, 2, 7, 33, 100])
def test_naive_lu_inverse_matches_lapack(oracle, n):
    rng = np.random.default_rng(100 + n)
    A = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    Ai = oracle.inverse(A)
    ref = np.linalg.inv(A)
    assert np.max(np.abs(Ai - ref)) <= 1e-10 * np.max(np.abs(ref))
    assert np.max(np.abs(A @ Ai - np.eye(n))) < 1e-10


def test_naive_lu_needs_and_uses_pivoting(oracle):
    # leading zero pivot: fails without row exchanges
    A = np.array([[0, 1, 2], [1, 0, 3], [4, 5, 6]], dtype=complex) + 1j * np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]])
    assert np.allclose(oracle.inverse(A), np.linalg.inv(A), atol=1e-13)
    # non-symmetric input: a transposed operand in the solve would show
    B = np.triu(np.ones((5, 5))) * (1 + 2j) + np.diag(np.arange(5))
    assert np.allclose(oracle.inverse(B), np.linalg.inv(B), atol=1e-13)


def test_singular_is_reported(oracle):
    with pytest.raises(oracle.OracleError) as e:
        oracle.inverse(np.zeros((3, 3), dtype=complex))
    assert e.value.code == -5


def test_naive_matmul_matches_lapack(oracle):
    rng = np.random.default_rng(7)
    A = rng.standard_normal((37, 37)) + 1j * rng.standard_normal((37, 37))
    B = rng.standard_normal((37, 37)) + 1j * rng.standard_normal((37, 37))
    assert np.max(np.abs(oracle.matmul(A, B) - A @ B)) < 1e-12


# ----------------------------------------------------------------------------------------
# Lead surface Green's function (A2)
# ----------------------------------------------------------------------------------------

@pytest.mark.parametrize("M,L,E", [(6, 4, 0.3), (6, 5, -1.1), (20, 40, 0.5), (20, 40, 2.0), (20, 41, 0.05), (7, 3, 0.9)])
def test_lead_surface_is_the_fixed_point_of_the_semi_infinite_chain(oracle, M, L, E):
    """g(surface) = (z - H_c - V_a g' V_a)^-1 with g' = (z - H_c - V_b g V_b)^-1 (period 2 slices)."""
    z = E + 1j * ETA
    Hc = slice_H(M, np.zeros(M), T_HOP)
    for side, (ia, ib) in ((+1, (L, L + 1)), (-1, (-2, -1))):
        g, it = oracle.lead_surface(M, L, T_HOP, E, ETA, side)
        Va, Vb = np.diag(T_HOP * mask(ia, M)), np.diag(T_HOP * mask(ib, M))
        gp = np.linalg.inv(z * np.eye(M) - Hc - Vb @ g @ Vb)
        g2 = np.linalg.inv(z * np.eye(M) - Hc - Va @ gp @ Va)
        assert np.max(np.abs(g - g2)) < 1e-6 * max(1.0, np.max(np.abs(g)))  # fixed point is marginally stable in-band
        assert np.max(np.abs(g - g.T)) < 1e-10            # complex symmetric
        assert 1 <= it <= 64
        # retarded: -Im g is positive semi-definite
        w = np.linalg.eigvalsh(1j * (g - g.conj().T))
        assert w.min() > -1e-9


@pytest.mark.parametrize("M", [4, 10, 20, 33])
def test_lead_block_form_equals_cell_form(oracle, M):
    for L in (6, 7):
        for E in (-2.2, -0.4, 0.013, 1.3):
            for side in (+1, -1):
                g0, it0 = oracle.lead_surface(M, L, T_HOP, E, ETA, side, oracle.LEAD_CELL)
                g1, it1 = oracle.lead_surface(M, L, T_HOP, E, ETA, side, oracle.LEAD_BLOCK)
                assert np.max(np.abs(g0 - g1)) < 1e-10 * max(1.0, np.max(np.abs(g0)))


def test_self_energy_structure(oracle):
    M, L, E = 20, 40, 0.8
    SL, _ = oracle.lead_self_energy(M, L, None, T_HOP, E, ETA, -1)
    SR, _ = oracle.lead_self_energy(M, L, None, T_HOP, E, ETA, +1)
    # support: only rows/cols with m_{-1}=1 (j odd) resp. m_{L-1}=1
    mL, mR = mask(-1, M), mask(L - 1, M)
    assert np.all(SL[mL == 0, :] == 0) and np.all(SL[:, mL == 0] == 0)
    assert np.all(SR[mR == 0, :] == 0) and np.all(SR[:, mR == 0] == 0)
    assert np.max(np.abs(SL - SL.T)) < 1e-12
    # even L: both leads see the same bond parity, Sigma_R = Sigma_L
    assert np.max(np.abs(SL - SR)) < 1e-11
    # odd L: Sigma_R = J Sigma_L J (row reversal), M even
    SR_odd, _ = oracle.lead_self_energy(M, L + 1, None, T_HOP, E, ETA, +1)
    assert np.max(np.abs(SR_odd - SL[::-1, ::-1])) < 1e-11
    # Gamma = i(Sigma - Sigma^dagger) >= 0
    assert np.linalg.eigvalsh(1j * (SL - SL.conj().T)).min() > -1e-10


# ----------------------------------------------------------------------------------------
# End to end on the clean ribbon: closed form (configs[0]) and the paper's integer steps
# ----------------------------------------------------------------------------------------

def test_config0_matches_closed_form(oracle):
    w = inputs.config0()
    T = oracle.transmission_batch(w.onsite[0], None, w.t, w.energies, w.eta)
    for E, Tk in zip(w.energies, T):
        Tc, n_open, dist = closed_form_T(w.M, w.L, E)
        assert dist > 1e-4, "grid point on a subband edge"
        assert abs(Tk - Tc) < 1e-8, (E, Tk, Tc)          # BASELINE.json:north_star "to 1e-8"
        assert -1e-12 <= Tk <= n_open + 1e-9             # bounds (Q19)
    # bipartite symmetry T(E) = T(-E) on the 32 mirror pairs
    assert np.max(np.abs(T - T[::-1])) < 1e-9


def test_paper_integer_steps_at_small_eta(oracle):
    """the ideal ribbon shows "a step-like dependence with the conductance being a
    multiple of 2e^2/h".  With eta = 1e-12 the absorption exp(-2 eta L/v) is below 1e-8."""
    w = inputs.config0()
    steps = np.loadtxt(os.path.join(GOLDEN, "clean_M20_channel_counts.txt"))
    T = oracle.transmission_batch(w.onsite[0], None, w.t, steps[:, 0], 1e-12)
    assert np.max(np.abs(T - steps[:, 1])) < 1e-8
    assert np.max(np.abs(T - np.round(T))) < 1e-8


def test_clean_M244_channel_counts_and_gap(oracle):
    """30 nm ribbon of the paper: semiconducting, N_ch from the closed form."""
    M, L = 244, 6
    on = np.zeros((L, M))
    E = np.array([0.01, 0.05, 0.5])
    T = oracle.transmission_batch(on, None, T_HOP, E, ETA, method=oracle.LEAD_BLOCK)
    cf = [closed_form_T(M, L, e) for e in E]
    assert [c[1] for c in cf] == [0, 2, 16]
    assert T[0] < 1e-2 and T[0] >= 0          # inside the gap: evanescent only (short L -> not yet tiny)
    assert abs(T[1] - cf[1][0]) < 1e-8 and abs(T[2] - cf[2][0]) < 1e-8


# ----------------------------------------------------------------------------------------
# Recursion == definition (Eq. 4-5 reach exactly Eq. 1), incl. vacancies
# ----------------------------------------------------------------------------------------

@pytest.mark.parametrize("M,L", [(2, 1), (3, 2), (4, 3), (5, 4), (6, 7), (8, 5), (7, 1)])
def test_recursion_equals_definition(oracle, M, L):
    rng = np.random.default_rng(1000 * M + L)
    on = rng.uniform(-0.5, 0.5, size=(L, M))
    for E in (-1.7, 0.21, 0.9):
        gL, _ = oracle.lead_surface(M, L, T_HOP, E, ETA, -1)
        gR, _ = oracle.lead_surface(M, L, T_HOP, E, ETA, +1)
        T_def = definition_T(on, None, T_HOP, E, ETA, gL, gR)
        T_rec = oracle.transmission(on, None, T_HOP, E, ETA)
        T_bf, T_bf_rl = oracle.transmission_brute(on, None, T_HOP, E, ETA)
        assert abs(T_rec - T_def) < 1e-11 * max(1, T_def)
        assert abs(T_bf - T_def) < 1e-11 * max(1, T_def)
        assert abs(T_bf_rl - T_def) < 1e-11 * max(1, T_def)     # reciprocity of the definition


def test_vacancy_is_a_deleted_site(oracle):
    """Q15: hoppings zeroed + on-site 1e3 eV  ==  the site removed from the matrix."""
    M, L = 14, 5         # M + 1 = 15 divisible by 3: metallic, T = O(1) at the energies below
    rng = np.random.default_rng(42)
    on = rng.uniform(-0.1, 0.1, size=(L, M))
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[0, 1] = vac[2, 0] = vac[4, 12] = vac[3, 13] = 1   # incl. sites bonded to both leads
    on[vac != 0] = inputs.VACANCY_ONSITE
    for E in (-1.8, 0.37, 2.4):
        gL, _ = oracle.lead_surface(M, L, T_HOP, E, ETA, -1)
        gR, _ = oracle.lead_surface(M, L, T_HOP, E, ETA, +1)
        T_del = definition_T(on, vac, T_HOP, E, ETA, gL, gR, delete_vacant=True)
        T_iso = definition_T(on, vac, T_HOP, E, ETA, gL, gR, delete_vacant=False)
        T_rec = oracle.transmission(on, vac, T_HOP, E, ETA)
        T_bf, _ = oracle.transmission_brute(on, vac, T_HOP, E, ETA)
        assert abs(T_iso - T_del) < 1e-12
        assert abs(T_rec - T_del) < 1e-11
        assert abs(T_bf - T_del) < 1e-11
        # and it differs from the ribbon without vacancies (the flags are not ignored)
        on_clean = np.where(vac != 0, 0.0, on)
        assert T_rec > 1e-3 and abs(oracle.transmission(on_clean, None, T_HOP, E, ETA) - T_rec) > 1e-3


# ----------------------------------------------------------------------------------------
# Invariants on disordered ribbons (the only hold on "parity unpinned" configs)
# ----------------------------------------------------------------------------------------

def test_reciprocity_and_symmetries(oracle):
    M, L = 20, 30
    on = inputs.anderson(M, L, 0.25, 77)
    E = np.array([-1.3, -0.2, 0.05, 0.6, 1.9])
    T = oracle.transmission_batch(on, None, T_HOP, E, ETA)
    for k, e in enumerate(E):
        T_rl = oracle.transmission(on, None, T_HOP, e, ETA, direction=1)
        assert abs(T[k] - T_rl) < 1e-11 * max(1, T[k])                       # T_LR = T_RL
        T_neg = oracle.transmission(-on, None, T_HOP, -e, ETA)
        assert abs(T[k] - T_neg) < 1e-11 * max(1, T[k])                      # T(E; eps) = T(-E; -eps)
        T_t = oracle.transmission(on, None, -T_HOP, e, ETA)
        assert abs(T[k] - T_t) < 1e-11 * max(1, T[k])                        # t -> -t gauge (Q12)
        n_open = closed_form_T(M, L, e)[1]
        assert -1e-12 <= T[k] <= n_open + 1e-9                               # Q19
        assert T[k] < n_open - 1e-6                                          # disorder does scatter


def test_im_trace_is_zero_and_iterations(oracle):
    w = inputs.config0()
    T, im, its = oracle.transmission(w.onsite[0], None, w.t, 0.4, w.eta, full=True)
    assert abs(im) < 1e-12
    assert 30 <= its[0] <= 45 and 30 <= its[1] <= 45     # ~log2(|t|/eta)+5


def test_sweep_state_is_block_of_left_connected_inverse(oracle):
    """g_i and P_i after i+1 slices are the (i,i) and (i,0) blocks of the inverse of the
    left-connected device truncated after slice i (no right lead)."""
    M, L, n = 5, 6, 4
    rng = np.random.default_rng(3)
    on = rng.uniform(-0.3, 0.3, size=(L, M))
    E = 0.7
    g, P = oracle.sweep_state(on, None, T_HOP, E, ETA, n)
    gL, _ = oracle.lead_surface(M, L, T_HOP, E, ETA, -1)
    N = M * n
    H = np.zeros((N, N), dtype=complex)
    for i in range(n):
        H[i * M:(i + 1) * M, i * M:(i + 1) * M] = slice_H(M, on[i], T_HOP)
        if i + 1 < n:
            H[i * M:(i + 1) * M, (i + 1) * M:(i + 2) * M] = np.diag(T_HOP * mask(i, M))
            H[(i + 1) * M:(i + 2) * M, i * M:(i + 1) * M] = np.diag(T_HOP * mask(i, M))
    mL = T_HOP * mask(-1, M)
    H[:M, :M] += mL[:, None] * gL * mL[None, :]
    G = np.linalg.inv((E + 1j * ETA) * np.eye(N) - H)
    assert np.max(np.abs(g - G[N - M:, N - M:])) < 1e-12
    assert np.max(np.abs(P - G[N - M:, :M])) < 1e-12


# ----------------------------------------------------------------------------------------
# Generators
# ----------------------------------------------------------------------------------------

def test_generators_are_seeded_and_shaped():
    w = inputs.config1(L=10, n_E=8)
    assert w.onsite.shape == (4, 10, 128) and np.abs(w.onsite).max() <= 0.25
    assert np.array_equal(w.onsite, inputs.config1(L=10, n_E=8).onsite)
    assert not np.array_equal(w.onsite[0], w.onsite[1])
    w4 = inputs.config4(M=64, L=50)
    assert w4.vacancy.shape == (1, 50, 64)
    assert w4.vacancy[0][:, 1:-1].sum() == 0 and 0 < w4.vacancy.sum() < 30
    assert np.all(w4.onsite[w4.vacancy != 0] == inputs.VACANCY_ONSITE)
    w3 = inputs.config3(L=4)
    assert w3.n_E == 1024 and w3.energies[0] == -1.0 and w3.energies[511] == 1.0 and abs(w3.energies[512] + 0.05) < 1e-15
    assert 0.0 not in w3.energies            # even counts never sample E = 0 (Q7)


# ----------------------------------------------------------------------------------------
# The 80-bit evaluator behind tests/golden/near_neutrality_ld.txt (neither oracle nor CUDA), pinned both ways
# ----------------------------------------------------------------------------------------

def test_extended_precision_evaluator_matches_oracle_and_closed_form(oracle):
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_near_neutrality_ld", os.path.join(GOLDEN, "make_near_neutrality_ld.py"))
    ld = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(ld)
    # disordered, vacancies, odd M and odd L, away from E = 0: the oracle is accurate there
    M, L = 9, 7
    on = inputs.anderson(M, L, 0.3, 31)
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[0, 1] = vac[3, 0] = vac[L - 1, 4] = 1
    for E in (-1.3, 0.21, 0.9):
        T_or = oracle.transmission_batch(on, vac, T_HOP, np.array([E]), ETA)[0]
        assert abs(ld.transmission_ld(on, vac, T_HOP, E, ETA) - T_or) < 1e-11, E
    # clean metallic ribbon at |E| = 1e-5 eV: closed form
    M, L = 8, 6
    Tc = closed_form_T(M, L, 1e-5)[0]
    assert abs(ld.transmission_ld(np.zeros((L, M)), None, T_HOP, 1e-5, ETA) - Tc) < 1e-13


def test_near_neutrality_golden_is_consistent_with_the_oracle(oracle):
    """Stored 80-bit values vs the oracle: equal to 1e-9 where the oracle is accurate (|E| >= 1e-3 eV), and within the
    oracle's documented loss (< 1e-7) below."""
    path = os.path.join(GOLDEN, "near_neutrality_ld.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    assert len(rows) == 32
    for case in ("clean_M20", "clean_M20_vacancy"):
        w = inputs.near_neutrality(case)
        vac = None if w.vacancy is None else w.vacancy[0]
        T_or = oracle.transmission_batch(w.onsite[0], vac, w.t, w.energies, w.eta)
        T_ld = np.array([float(r[3]) for r in rows if r[0] == case])
        assert np.all(np.abs(T_or - T_ld) <= 1e-9), (case, np.abs(T_or - T_ld))


# ----------------------------------------------------------------------------------------
# O9: local density of states (diagonal blocks of the connected Green's function), SURVEY.md 8(f) F-4
# ----------------------------------------------------------------------------------------

def definition_ldos(onsite, vac, t, E, eta, gL, gR):
    """-(1/pi) Im diag of Eq. 1 written out with numpy: the whole device matrix, inverted at once."""
    L, M = onsite.shape
    N = M * L
    isvac = np.zeros((L, M), dtype=bool) if vac is None else vac.astype(bool)
    A = (E + 1j * eta) * np.eye(N, dtype=complex)
    for i in range(L):
        A[i * M:(i + 1) * M, i * M:(i + 1) * M] -= slice_H(M, onsite[i], t, isvac[i])
        if i + 1 < L:
            m = mask(i, M) * (~isvac[i]) * (~isvac[i + 1])
            A[i * M:(i + 1) * M, (i + 1) * M:(i + 2) * M] -= np.diag(t * m)
            A[(i + 1) * M:(i + 2) * M, i * M:(i + 1) * M] -= np.diag(t * m)
    mL = mask(-1, M) * (~isvac[0])
    mR = mask(L - 1, M) * (~isvac[L - 1])
    A[:M, :M] -= (t * mL)[:, None] * gL * (t * mL)[None, :]
    A[N - M:, N - M:] -= (t * mR)[:, None] * gR * (t * mR)[None, :]
    return (-np.diag(np.linalg.inv(A)).imag / np.pi).reshape(L, M)


@pytest.mark.parametrize("M,L", [(4, 1), (5, 2), (6, 7), (9, 6)])
def test_ldos_recursion_equals_definition(oracle, M, L):
    """The two-pass recursion against the full inverse, with disorder, vacancies (incl. both end slices), odd M and L."""
    on = inputs.anderson(M, L, 0.4, 50 + M)
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[0, 1] = 1
    if L > 2:
        vac[L // 2, 0] = vac[L - 1, M - 2] = 1
    on[vac != 0] = inputs.VACANCY_ONSITE
    E = np.array([-1.7, -0.3, 0.45, 1.2])
    for eta in (1e-3, 1e-6):
        got = oracle.ldos_batch(on, vac, T_HOP, E, eta)
        for k, e in enumerate(E):
            gL, _ = oracle.lead_surface(M, L, T_HOP, e, eta, -1)
            gR, _ = oracle.lead_surface(M, L, T_HOP, e, eta, +1)
            ref = definition_ldos(on, vac, T_HOP, e, eta, gL, gR)
            assert np.max(np.abs(got[k] - ref)) <= 1e-10 * max(1.0, np.max(np.abs(ref))), (M, L, e, eta)


def test_ldos_closed_forms_and_invariants(oracle):
    M, L, eta = 8, 6, 1e-3
    E = np.array([-0.9, 0.37])
    # a vacancy is an isolated level at its on-site energy: G = 1 / (z - eps), LDOS = (eta / pi) / ((E - eps)^2 + eta^2)
    on = np.zeros((L, M))
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[2, 3] = 1
    on[2, 3] = 0.5
    got = oracle.ldos_batch(on, vac, T_HOP, E, eta)
    for k, e in enumerate(E):
        assert abs(got[k, 2, 3] - (eta / np.pi) / ((e - 0.5) ** 2 + eta ** 2)) < 1e-12
    # clean ribbon between clean leads = infinite ribbon: LDOS >= 0, periodic with the two-slice cell, and (zero on-site
    # energies, bipartite lattice) the same at E and -E
    clean = oracle.ldos_batch(np.zeros((L, M)), None, T_HOP, np.array([0.8, -0.8, 1.9]), eta)
    assert np.all(clean > 0)
    assert np.max(np.abs(clean[:, 2:] - clean[:, :-2])) < 1e-9 * np.max(clean)
    assert np.max(np.abs(clean[0] - clean[1])) < 1e-12 * np.max(clean)
    # one-dimensional check of the scale: M = 2 ... the integrated weight of a site is 1 (Lorentzian tails of width eta):
    # a single isolated device site (both neighbours vacant) integrates to 1
    on1 = np.zeros((3, 3))
    v1 = np.ones((3, 3), dtype=np.uint8)
    v1[1, 1] = 0                       # only the centre site is not a vacancy; every bond to it is cut
    grid = np.linspace(-0.2, 0.2, 4001)
    w = oracle.ldos_batch(on1, v1, T_HOP, grid, 5e-3)[:, 1, 1]
    assert abs(np.trapezoid(w, grid) - 2 / np.pi * np.arctan(0.2 / 5e-3)) < 1e-6


# ----------------------------------------------------------------------------------------
# O10: the paper's own Eq. 4 form, double and single precision (SURVEY.md 8(c) "Precision finding")
# ----------------------------------------------------------------------------------------

def test_eq4_form_equals_direct_form_in_double(oracle):
    """(1 - G0 V G V)^-1 G0 = (z - H - V G V)^-1: the two forms of Eq. 4 agree to rounding away from the levels of the
    isolated slices (disorder, vacancies on both end slices, odd M and L)."""
    M, L = 9, 7
    on = inputs.anderson(M, L, 0.3, 31)
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[0, 1] = vac[3, 0] = vac[L - 1, 4] = 1
    on[vac != 0] = inputs.VACANCY_ONSITE
    E = np.array([-1.3, -0.37, 0.21, 0.9])
    T_direct = oracle.transmission_batch(on, vac, T_HOP, E, ETA)
    T_eq4 = oracle.transmission_eq4_batch(on, vac, T_HOP, E, ETA, use_float=False)
    assert np.max(np.abs(T_eq4 - T_direct)) < 1e-10


def test_eq4_form_in_single_precision_is_single_precision(oracle):
    """The float sweep (own float LU and matmul) lands within single-precision distance of the double one on a short benign
    ribbon -- a wrong index or sign in the float routines would be O(1) off -- and is not the double result."""
    w = inputs.config0(M=20, L=12, n_E=6)
    E = w.energies + 0.0131
    T_d = oracle.transmission_eq4_batch(w.onsite[0], None, w.t, E, w.eta, use_float=False)
    T_f = oracle.transmission_eq4_batch(w.onsite[0], None, w.t, E, w.eta, use_float=True)
    d = np.abs(T_f - T_d)
    assert np.all(np.isfinite(T_f)) and d.max() < 1e-3 and d.max() > 1e-9
