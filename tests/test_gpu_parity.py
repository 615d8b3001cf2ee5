"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerance (BASELINE.json:north_star): complex128 |dT| <= 1e-9 * max(1, T).
"""
import os

import numpy as np
import pytest

from paper_1107_5300_b200 import inputs

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def rgf():
    from paper_1107_5300_b200 import binding
    return binding


@pytest.fixture()
def plan(rgf):
    with rgf.Plan(0) as p:
        yield p


FORMS = [0, 1, 2]          # RGF_FORM_DENSE, RGF_FORM_HALF (fused kernel for M <= 256), RGF_FORM_HALF_STEPWISE (include/rgf.h)


@pytest.fixture(params=FORMS, ids=["dense", "half", "half_stepwise"])
def fplan(rgf, request):
    """A plan in each formulation of the sweep."""
    with rgf.Plan(0) as p:
        rgf.rgf_set_formulation(p.handle, request.param)
        p.form = request.param
        yield p


def tol(T):
    return 1e-9 * np.maximum(1.0, np.abs(T))


# ---- A4: the batched inverse on its own -----------------------------------------------------

@pytest.mark.parametrize("n,batch", [(1, 3), (5, 4), (20, 7), (32, 2), (33, 3), (64, 2), (100, 5), (244, 6), (256, 2), (257, 2), (300, 2), (301, 3), (512, 2), (515, 1), (600, 1), (1100, 1), (1101, 1), (2048, 1)])
def test_inverse_batched_matches_oracle_and_lapack(rgf, plan, oracle, n, batch):
    rng = np.random.default_rng(n * 31 + batch)
    A = rng.standard_normal((batch, n, n)) + 1j * rng.standard_normal((batch, n, n))
    A[0] += np.diag(np.zeros(n))
    if n >= 5:
        A[-1, 0, 0] = 0.0            # forces a row exchange in the first column
        A[-1, 3, 3] = 0.0
    out = np.empty_like(A)
    rgf.rgf_inverse_batched(plan.handle, n, batch, A, out)
    for b in range(batch):
        ref = np.linalg.inv(A[b])
        scale = np.max(np.abs(ref))
        assert np.max(np.abs(out[b] - ref)) < 1e-9 * scale, (b, np.max(np.abs(out[b] - ref)) / scale)
        assert np.max(np.abs(A[b] @ out[b] - np.eye(n))) < 1e-8
    if n <= 100:
        assert np.max(np.abs(out[0] - oracle.inverse(A[0]))) < 1e-9 * np.max(np.abs(out[0]))


def test_inverse_of_actual_slice_matrix(rgf, plan, oracle):
    """A_i = z - H_i - Sigma of a disordered M=244 slice: complex symmetric, tiny imaginary part."""
    M = 244
    rng = np.random.default_rng(5)
    on = rng.uniform(-0.1, 0.1, M)
    A = np.zeros((3, M, M), dtype=complex)
    for b, E in enumerate((0.013, 0.5, -0.97)):
        A[b] = np.diag(E + 1e-9j - on) - np.diag(np.full(M - 1, -2.7), 1) - np.diag(np.full(M - 1, -2.7), -1)
    out = np.empty_like(A)
    rgf.rgf_inverse_batched(plan.handle, M, 3, A, out)
    for b in range(3):
        ref = oracle.inverse(A[b])
        assert np.max(np.abs(out[b] - ref)) < 1e-9 * np.max(np.abs(ref))


def test_singular_matrix_is_reported(rgf, plan):
    A = np.zeros((2, 8, 8), dtype=complex)
    A[0] = np.eye(8)
    out = np.empty_like(A)
    with pytest.raises(rgf.RgfError) as e:
        rgf.rgf_inverse_batched(plan.handle, 8, 2, A, out)
    assert e.value.code == rgf.RGF_ESINGULAR


# ---- A2: lead self-energies -----------------------------------------------------------------

@pytest.mark.parametrize("method", [0, 1, 2], ids=["cell_dense", "cell_schur", "mode_space"])
@pytest.mark.parametrize("M,L", [(20, 40), (20, 41), (7, 5), (21, 9), (21, 10), (64, 10)])
def test_lead_self_energy_matches_oracle(rgf, plan, oracle, M, L, method):
    rgf.rgf_set_lead_method(plan.handle, method)
    E = np.array([-2.0, -0.4, 0.013, 0.8, 1.7])
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[0, 1] = 1
    vac[L - 1, 2 if (L - 1) % 2 == 0 else 3] = 1
    on = np.zeros((L, M))
    plan.set_device(on, -2.7, vac)
    for side in (-1, +1):
        S = np.empty((len(E), M, M), dtype=complex)
        it = rgf.rgf_lead_self_energy(plan.handle, 0, E, len(E), 1e-9, side, S)
        assert (it == 0) if method == 2 else (20 <= it <= 64)
        for k, e in enumerate(E):
            ref, _ = oracle.lead_self_energy(M, L, vac, -2.7, e, 1e-9, side)
            assert np.max(np.abs(S[k] - ref)) < 1e-9 * max(1.0, np.max(np.abs(ref))), (side, e)


def test_lead_self_energy_mode_space_at_paper_width(rgf, plan, oracle):
    """M = 244 (the headline width): the mode-space closed form (default) against the oracle's Sancho-Rubio cell form,
    element by element, at two energies (the naive 488 x 488 decimation takes about a minute per energy)."""
    from concurrent.futures import ThreadPoolExecutor
    M, L = 244, 6
    E = np.array([-0.6213, 0.4637])          # 0.4637 eV: where the block decimation once diverged
    plan.set_device(np.zeros((L, M)), -2.7)
    S = np.empty((2, M, M), dtype=complex)
    assert rgf.rgf_lead_self_energy(plan.handle, 0, E, 2, 1e-9, -1, S) == 0
    with ThreadPoolExecutor(2) as ex:
        refs = list(ex.map(lambda e: oracle.lead_self_energy(M, L, None, -2.7, e, 1e-9, -1)[0], E))
    for k in range(2):
        assert np.max(np.abs(S[k] - refs[k])) < 1e-9 * max(1.0, np.max(np.abs(refs[k]))), (E[k], np.max(np.abs(S[k] - refs[k])))


def test_lead_sigma_is_masked_on_the_device(rgf, plan, oracle):
    """Sigma = t^2 m' (.) g (.) m' with a vacancy on the end slice: the rows / columns of the vacant atom are zero."""
    M, L = 20, 6
    vac = np.zeros((L, M), dtype=np.uint8)
    vac[0, 3] = 1
    plan.set_device(np.zeros((L, M)), -2.7, vac)
    E = np.array([0.37])
    S = np.empty((1, M, M), dtype=complex)
    rgf.rgf_lead_self_energy(plan.handle, 0, E, 1, 1e-9, -1, S)
    ref, _ = oracle.lead_self_energy(M, L, vac, -2.7, 0.37, 1e-9, -1)
    assert np.all(S[0][3, :] == 0) and np.all(S[0][:, 3] == 0) and np.all(S[0][0::2, :] == 0)
    assert np.max(np.abs(S[0] - ref)) < 1e-9 * np.max(np.abs(ref))


# ---- A3-A5: state of the sweep ---------------------------------------------------------------

@pytest.mark.parametrize("M,L,ns", [(20, 12, 1), (20, 12, 2), (20, 12, 7), (21, 9, 9), (64, 6, 5)])
def test_sweep_state_matches_oracle(rgf, fplan, oracle, M, L, ns):
    plan = fplan
    on = inputs.anderson(M, L, 0.25, 99 + M)
    plan.set_device(on, -2.7)
    E = np.array([-1.1, 0.07, 0.9])
    g = np.empty((3, M, M), dtype=complex)
    P = np.empty((3, M, M), dtype=complex)
    rgf.rgf_sweep_state(plan.handle, 0, E, 3, 1e-9, rgf.RGF_C128, ns, g, P)
    for k, e in enumerate(E):
        g0, P0 = oracle.sweep_state(on, None, -2.7, e, 1e-9, ns)
        if plan.form != rgf.RGF_FORM_DENSE:       # only the F_i x F_i block of G_ii exists in this formulation
            hg = ~np.isnan(g[k].real)
            fr = (np.arange(M) % 2) == ((ns - 1) % 2)
            assert np.array_equal(hg, np.outer(fr, fr))
            assert np.max(np.abs(g[k][hg] - g0[hg])) < 1e-9 * np.max(np.abs(g0))
        else:
            assert np.max(np.abs(g[k] - g0)) < 1e-9 * np.max(np.abs(g0))
        have = ~np.isnan(P[k].real)
        rows = (np.arange(M) % 2) == ((ns - 1) % 2)
        cols = (np.arange(M) % 2) == 1
        assert np.array_equal(have, np.outer(rows, cols))
        assert np.max(np.abs(P[k][have] - P0[have])) < 1e-9 * max(1e-300, np.max(np.abs(P0)))


# ---- end to end ----------------------------------------------------------------------------

def test_config0_matches_oracle_and_closed_form(rgf, fplan, oracle):
    plan = fplan
    from test_oracle_pins import closed_form_T
    w = inputs.config0()
    plan.set_device(w.onsite, w.t)
    T = plan.transmission(w.energies, w.eta)[0]
    T_or = oracle.transmission_batch(w.onsite[0], None, w.t, w.energies, w.eta)
    assert np.all(np.abs(T - T_or) <= tol(T_or)), np.max(np.abs(T - T_or))
    for e, tk in zip(w.energies, T):
        assert abs(tk - closed_form_T(w.M, w.L, e)[0]) < 1e-8
    assert plan.stats()["launches"] > 0


@pytest.mark.parametrize("M,L,W", [(2, 3, 0.2), (3, 4, 0.2), (20, 1, 0.2), (20, 2, 0.2), (21, 17, 0.3), (50, 33, 0.25), (128, 24, 0.25)])
def test_disordered_small_matches_oracle(rgf, fplan, oracle, M, L, W):
    plan = fplan
    on = inputs.anderson(M, L, W, 1000 + M + L)
    E = np.linspace(-1.0, 1.0, 8)
    plan.set_device(on, -2.7)
    T = plan.transmission(E, 1e-9)[0]
    T_or = oracle.transmission_batch(on, None, -2.7, E, 1e-9)
    assert np.all(np.abs(T - T_or) <= tol(T_or)), np.max(np.abs(T - T_or))


def test_batched_devices_vacancies_and_cohorts(rgf, fplan, oracle):
    plan = fplan
    """4 devices batched (configs[1] shape, reduced), one with edge vacancies; ragged cohorts."""
    M, L = 32, 20
    on = np.stack([inputs.anderson(M, L, 0.25, s) for s in (1107, 1108, 1109)])
    vac = np.zeros((3, L, M), dtype=np.uint8)
    vac[2] = inputs.edge_vacancies(M, L, 0.3, 5303)
    vac[2, 0, 1] = 1
    on[vac != 0] = inputs.VACANCY_ONSITE
    E = np.linspace(-1.0, 1.0, 8)          # even count: E = 0 (a resonance of the isolated lead cell) is not sampled
    plan.set_device(on, -2.7, vac)
    T_ref = np.stack([oracle.transmission_batch(on[d], vac[d], -2.7, E, 1e-9) for d in range(3)])
    for cohort in (0, 5, 21, 4):
        rgf.rgf_set_cohort(plan.handle, cohort)
        T = plan.transmission(E, 1e-9)
        assert T.shape == (3, 8)
        assert np.all(np.abs(T - T_ref) <= tol(T_ref)), (cohort, np.max(np.abs(T - T_ref)))


def test_device_pointers(rgf, plan, oracle):
    import torch
    w = inputs.config0(n_E=16)
    plan.set_device(w.onsite, w.t)
    E = torch.tensor(w.energies, dtype=torch.float64, device="cuda")
    T = torch.empty(16, dtype=torch.float64, device="cuda")
    rgf.rgf_transmission(plan.handle, E, 16, w.eta, rgf.RGF_C128, T)
    T_or = oracle.transmission_batch(w.onsite[0], None, w.t, w.energies, w.eta)
    assert np.all(np.abs(T.cpu().numpy() - T_or) <= tol(T_or))


def test_errors(rgf, plan):
    E = np.array([0.1])
    T = np.empty(1)
    with pytest.raises(rgf.RgfError) as e:
        rgf.rgf_transmission(plan.handle, E, 1, 1e-9, rgf.RGF_C128, T)
    assert e.value.code == rgf.RGF_ESTATE
    plan.set_device(np.zeros((4, 6)), -2.7)
    for bad in (dict(eta=0.0), dict(eta=-1.0)):
        with pytest.raises(rgf.RgfError) as e:
            rgf.rgf_transmission(plan.handle, E, 1, bad["eta"], rgf.RGF_C128, T)
        assert e.value.code == rgf.RGF_EINVAL
    with pytest.raises(rgf.RgfError) as e:
        rgf.rgf_transmission(plan.handle, np.array([np.nan]), 1, 1e-9, rgf.RGF_C128, T)
    assert e.value.code == rgf.RGF_EINVAL
    with pytest.raises(rgf.RgfError) as e:
        rgf.rgf_set_device(plan.handle, 1, 4, np.zeros((4, 1)), -2.7)
    assert e.value.code == rgf.RGF_EINVAL


# ---- complex64 sweep (configs[3] precision study; reading R13) ---------------------------

@pytest.mark.parametrize("M,L,W", [(20, 40, 0.0), (21, 17, 0.3), (64, 50, 0.1), (244, 30, 0.1)])
def test_c64_sweep_close_to_c128_and_oracle(rgf, plan, oracle, M, L, W):
    """north_star: the complex64 path stays within |dT| <= 1e-3 outside |E| < 0.1 eV."""
    on = inputs.anderson(M, L, W, 77 + M) if W > 0 else np.zeros((L, M))
    E = np.concatenate([np.linspace(-1.0, -0.1, 6), np.linspace(0.1, 1.0, 6)]) + 0.0037
    plan.set_device(on, -2.7)
    T128 = plan.transmission(E, 1e-9)[0]
    T64 = plan.transmission(E, 1e-9, precision=rgf.RGF_C64)[0]
    assert np.all(np.isfinite(T64))
    assert np.max(np.abs(T64 - T128)) <= 1e-3, np.abs(T64 - T128)
    assert np.max(np.abs(T64 - T128)) > 0.0            # it really ran in another precision
    if M <= 64:
        T_or = oracle.transmission_batch(on, None, -2.7, E, 1e-9)
        assert np.max(np.abs(T64 - T_or)) <= 1e-3


def test_c64_sweep_state_matches_oracle_to_single_precision(rgf, plan, oracle):
    M, L, ns = 50, 9, 6
    on = inputs.anderson(M, L, 0.25, 5)
    plan.set_device(on, -2.7)
    E = np.array([-0.8, 0.31])
    g = np.empty((2, M, M), dtype=complex)
    P = np.empty((2, M, M), dtype=complex)
    rgf.rgf_sweep_state(plan.handle, 0, E, 2, 1e-9, rgf.RGF_C64, ns, g, P)
    for k, e in enumerate(E):
        g0, P0 = oracle.sweep_state(on, None, -2.7, e, 1e-9, ns)
        hg = ~np.isnan(g[k].real)
        assert hg.sum() == (M // 2) ** 2
        assert np.max(np.abs(g[k][hg] - g0[hg])) < 2e-4 * np.max(np.abs(g0))
        hp = ~np.isnan(P[k].real)
        assert np.max(np.abs(P[k][hp] - P0[hp])) < 2e-4 * np.max(np.abs(P0))
        assert np.max(np.abs(g[k][hg] - g0[hg])) > 1e-12 * np.max(np.abs(g0))      # single precision, not double


def test_c64_needs_half_formulation(rgf, plan):
    plan.set_device(np.zeros((4, 6)), -2.7)
    rgf.rgf_set_formulation(plan.handle, rgf.RGF_FORM_DENSE)
    with pytest.raises(rgf.RgfError) as e:
        plan.transmission(np.array([0.3]), 1e-9, precision=rgf.RGF_C64)
    assert e.value.code == rgf.RGF_EUNSUPPORTED


def test_fused_kernel_unit_rounds(rgf, plan, oracle):
    """The fused kernel runs in rounds of units (matrix, 64 half-steps) when there are more matrices than CTA slots: force
    3 slots for 2 devices x 5 energies and 3 chunks of half-steps, so that every matrix is resumed twice from the state
    (X, W, perm) it left in HBM, by a different CTA each time."""
    M, L = 21, 70
    on = np.stack([inputs.anderson(M, L, 0.3, 41), inputs.anderson(M, L, 0.3, 42)])
    E = np.array([-1.3, -0.41, 0.07, 0.66, 1.9])
    plan.set_device(on, -2.7)
    T_ref = np.stack([oracle.transmission_batch(on[d], None, -2.7, E, 1e-9) for d in range(2)])
    for slots in (3, 4, 0):
        rgf.rgf_set_cohort(plan.handle, slots)
        T = plan.transmission(E, 1e-9)
        assert np.all(np.abs(T - T_ref) <= tol(T_ref)), (slots, np.max(np.abs(T - T_ref)))
    rgf.rgf_set_cohort(plan.handle, 3)
    T = plan.transmission(E, 1e-9)
    st = plan.stats()
    assert st["cohort"] == 10                          # the fused kernel keeps the whole batch as one cohort ...
    assert st["launches_inverse_update"] == 10         # ... and runs ceil(10 matrices x 3 chunks / 3 slots) launches of units
    assert np.all(np.abs(T - T_ref) <= tol(T_ref))


def test_fused_state_across_unit_rounds_with_vacancies(rgf, plan, oracle):
    """State (g, P) of the fused kernel after 35 slices = 70 half-steps, i.e. two units, with 2 CTA slots for 3 energies: the B
    half-steps are assembled in place from the previous result through the row / column maps, which a matrix carries
    through HBM from one launch to the next; odd width (the two halves differ in size) and vacancies (masked rows / columns
    of the in-place assembly)."""
    M, L, ns = 21, 40, 35
    on = inputs.anderson(M, L, 0.3, 77)
    vac = inputs.edge_vacancies(M, L, 0.25, 13)
    on[vac != 0] = inputs.VACANCY_ONSITE
    E = np.array([-1.2, 0.31, 0.95])
    plan.set_device(on, -2.7, vac)
    rgf.rgf_set_cohort(plan.handle, 2)
    g = np.empty((3, M, M), dtype=complex)
    P = np.empty((3, M, M), dtype=complex)
    rgf.rgf_sweep_state(plan.handle, 0, E, 3, 1e-9, rgf.RGF_C128, ns, g, P)
    rgf.rgf_set_cohort(plan.handle, 0)
    for k, e in enumerate(E):
        g0, P0 = oracle.sweep_state(on, vac, -2.7, e, 1e-9, ns)
        hg = ~np.isnan(g[k].real)
        fr = (np.arange(M) % 2) == ((ns - 1) % 2)
        assert np.array_equal(hg, np.outer(fr, fr))
        assert np.max(np.abs(g[k][hg] - g0[hg])) < 1e-9 * np.max(np.abs(g0))
        have = ~np.isnan(P[k].real)
        assert np.array_equal(have, np.outer(fr, (np.arange(M) % 2) == 1))
        assert np.max(np.abs(P[k][have] - P0[have])) < 1e-9 * max(1e-300, np.max(np.abs(P0)))


@pytest.mark.parametrize("M,L", [(21, 9), (32, 12)])
def test_c64_with_vacancies_and_odd_width(rgf, plan, oracle, M, L):
    on = inputs.anderson(M, L, 0.2, 7 * M)
    vac = inputs.edge_vacancies(M, L, 0.3, 11)
    on[vac != 0] = inputs.VACANCY_ONSITE
    E = np.array([-1.4, -0.6, 0.35, 1.1])
    plan.set_device(on, -2.7, vac)
    T64 = plan.transmission(E, 1e-9, precision=rgf.RGF_C64)[0]
    T_or = oracle.transmission_batch(on, vac, -2.7, E, 1e-9)
    assert np.max(np.abs(T64 - T_or)) <= 1e-3, np.abs(T64 - T_or)


def test_lead_methods_agree_and_fall_back_near_t(rgf, plan, oracle):
    """RGF_LEAD_CELL_SCHUR eliminates half of the cell in closed form, resonant at E = +-t: such calls take the dense route."""
    M, L = 20, 40
    on = np.zeros((L, M))
    plan.set_device(on, -2.7)
    E = np.array([-2.7, -2.69, 0.5, 2.7])
    T_or = oracle.transmission_batch(on, None, -2.7, E, 1e-9)
    for method in (0, 1, 2):
        rgf.rgf_set_lead_method(plan.handle, method)
        T = plan.transmission(E, 1e-9)[0]
        assert np.all(np.abs(T - T_or) <= tol(T_or)), (method, np.abs(T - T_or))


def test_lead_methods_agree_at_paper_width(rgf, plan):
    """M = 244 at E = 0.4637 eV: the block decimation diverged there before beta = alpha^T was made structural
    (DESIGN.md section 5c); both lead routes must converge and give the same T on a short clean ribbon."""
    M, L = 244, 4
    plan.set_device(np.zeros((L, M)), -2.7)
    E = np.array([-0.4, 0.2549, 0.4637, 0.8])
    T = []
    for method in (0, 1, 2):
        rgf.rgf_set_lead_method(plan.handle, method)
        T.append(plan.transmission(E, 1e-9)[0])
        assert (plan.stats()["lead_iterations"] == 0) if method == 2 else (30 <= plan.stats()["lead_iterations"] <= 40)
    assert np.all(np.isfinite(T[0])) and np.all(np.isfinite(T[1])) and np.all(np.isfinite(T[2]))
    assert np.all(np.abs(T[0] - T[1]) <= 1e-9 * np.maximum(1.0, T[0])), np.abs(T[0] - T[1])
    assert np.all(np.abs(T[0] - T[2]) <= 1e-9 * np.maximum(1.0, T[0])), np.abs(T[0] - T[2])
    assert np.all(np.abs(T[0] - np.round(T[0])) < 1e-6)          # clean ribbon: integer channel count up to the eta deficit


# ---- near charge neutrality: conducting ribbons at |E| -> 0 -----------------------------

def near_neutrality_ld():
    """{case: T[8]} in 80-bit arithmetic, written by tests/golden/make_near_neutrality_ld.py (neither oracle nor CUDA)."""
    out = {}
    for line in open(os.path.join(GOLDEN, "near_neutrality_ld.txt")):
        if line.startswith("#"):
            continue
        c, k, e, tv = line.split()
        out.setdefault(c, {})[int(k)] = (float(e), float(tv))
    return out


@pytest.mark.parametrize("case", inputs.NEAR_NEUTRALITY_CASES)
def test_near_charge_neutrality_default_formulation(rgf, plan, oracle, case):
    """Metallic ribbons (M = 20 and M = 128: M + 1 divisible by 3, one open channel at |E| -> 0) in the DEFAULT formulation
    at |E| = 1e-2 ... 1e-5 eV.  The half-slice cut loses ~eps (t/E)^2 in a clean ribbon there, so the library must route such
    energies to the dense formulation by itself (rgf_set_guard default).  Element = each energy, tolerance 1e-9 max(1, T):
    against the oracle for |E| >= 1e-3 eV, and against the 80-bit values of tests/golden/near_neutrality_ld.txt at every
    energy (below 1e-3 eV the oracle's own lead decimation is off by up to 3e-8: make_near_neutrality_ld.py says why)."""
    from test_oracle_pins import closed_form_T
    w = inputs.near_neutrality(case)
    vac = None if w.vacancy is None else w.vacancy[0]
    plan.set_device(w.onsite, w.t, w.vacancy)
    T = plan.transmission(w.energies, w.eta)[0]
    st = plan.stats()
    ld = near_neutrality_ld()[case]
    T_ld = np.array([ld[k][1] for k in range(8)])
    assert np.array_equal(np.array([ld[k][0] for k in range(8)]), w.energies)
    err = np.abs(T - T_ld) / np.maximum(1.0, T_ld)
    assert np.all(err <= 1e-9), (case, err, st["guard_redone"])
    big = np.abs(w.energies) >= 1e-3
    T_or = oracle.transmission_batch(w.onsite[0], vac, w.t, w.energies[big], w.eta)
    assert np.all(np.abs(T[big] - T_or) <= 1e-9 * np.maximum(1.0, T_or)), (case, np.abs(T[big] - T_or))
    if case != "clean_M20_vacancy":
        assert np.all(T_ld > 0.05)                 # conducting: the absolute tolerance does not hide a relative error
    if case == "clean_M20":
        assert st["guard_redone"] >= 4             # |E| <= 1e-4 eV cannot be held by the half-slice formulation
        for e, tk in zip(w.energies, T):
            assert abs(tk - closed_form_T(w.M, w.L, e)[0]) < 1e-9
        # the guard is what makes it pass: without it the smallest |E| are off by more than the tolerance
        rgf.rgf_set_guard(plan.handle, 0.0)
        T_half = plan.transmission(w.energies, w.eta)[0]
        rgf.rgf_set_guard(plan.handle, 1e-10)
        assert plan.stats()["guard_redone"] == 0
        assert np.max(np.abs(T_half - T_ld)[-2:]) > 1e-9


def test_guard_indicator_tracks_the_resonance(rgf, plan):
    """G = |t| / (smallest pivot) of the clean metallic ribbon grows like |t / E| (the dangling-bond resonance sits at E = 0)."""
    M, L = 20, 40
    plan.set_device(np.zeros((L, M)), -2.7)
    E = np.array([0.3, 1e-2, 1e-3, 1e-4])
    rgf.rgf_set_guard(plan.handle, 1e30)           # record, never redo
    plan.transmission(E, 1e-9)
    G, Gmax = np.zeros(4), np.zeros(4)
    rgf.rgf_get_guard_indicators(plan.handle, G, Gmax, 4)
    rgf.rgf_set_guard(plan.handle, 1e-10)
    print("guard indicators", G, Gmax)
    assert G[0] < 50 and np.all(G[1:] > 0.2 * 2.7 / E[1:]) and np.all(G[1:] < 20 * 2.7 / E[1:])
    assert np.all(Gmax >= G * 0.99) and np.all(Gmax < 2.0 * G + 50)      # clean ribbon: every half-step has the same pivot


# ---- F-4: local density of states of the connected device (rgf_ldos) ---------------------------------------------------------

@pytest.mark.parametrize("M,L,W,with_vac", [(20, 12, 0.25, False), (21, 9, 0.3, True), (64, 10, 0.1, True), (20, 1, 0.2, False),
                                             (128, 7, 0.25, False), (300, 3, 0.1, True)])
def test_ldos_matches_oracle(rgf, plan, oracle, M, L, W, with_vac):
    """LDOS[i][j] = -(1/pi) Im G_ii[j][j] element by element against the oracle's two-pass recursion (itself pinned to the full
    inverse); two devices batched, eta = 1e-3 eV (a smooth LDOS).  Tolerance 1e-9 max(1, max LDOS)."""
    on = np.stack([inputs.anderson(M, L, W, 300 + M), inputs.anderson(M, L, W, 301 + M)])
    vac = None
    if with_vac:
        vac = np.zeros((2, L, M), dtype=np.uint8)
        vac[0, 0, 1] = vac[0, L - 1, 2] = vac[1, L // 2, 0] = 1
        on[vac != 0] = inputs.VACANCY_ONSITE
    E = np.array([-1.3, -0.2, 0.07, 0.9, 2.1])
    plan.set_device(on, -2.7, vac)
    got = plan.ldos(E, 1e-3)
    assert got.shape == (2, len(E), L, M)
    for d in range(2):
        ref = oracle.ldos_batch(on[d], None if vac is None else vac[d], -2.7, E, 1e-3)
        err = np.max(np.abs(got[d] - ref))
        assert err <= 1e-9 * max(1.0, np.max(np.abs(ref))), (M, L, d, err, np.max(np.abs(ref)))
    assert np.all(got > 0)
    assert plan.stats()["launches"] > 0


def test_ldos_device_pointers_and_chunks(rgf, plan, oracle):
    import torch
    M, L = 32, 8
    on = inputs.anderson(M, L, 0.2, 9)
    plan.set_device(on, -2.7)
    E = np.linspace(-1.0, 1.0, 6)
    E_dev = torch.tensor(E, dtype=torch.float64, device="cuda")
    out = torch.empty((1, 6, L, M), dtype=torch.float64, device="cuda")
    rgf.rgf_ldos(plan.handle, E_dev, 6, 2e-3, out)
    ref = oracle.ldos_batch(on, None, -2.7, E, 2e-3)
    assert np.max(np.abs(out.cpu().numpy()[0] - ref)) <= 1e-9 * max(1.0, np.max(ref))


@pytest.mark.parametrize("M,L", [(23, 41), (20, 5), (23, 4)])
def test_guard_pass_two_sided_sweep_odd_sizes(rgf, plan, oracle, M, L):
    """The guard's second pass sweeps the dense formulation from both leads and joins the two halves by Dyson's equation
    (run_dense_two_sided): odd M (the two sublattice blocks differ in size), odd L (g_R is a lead of its own, the halves
    differ in length), the shortest L it is used for, vacancies next to the junction.  Metallic clean ribbons (M + 1
    divisible by 3) at small |E| force every energy into that pass; closed form and oracle referee."""
    from test_oracle_pins import closed_form_T
    on = np.zeros((L, M))
    E = np.array([1e-3, -1e-3, 2e-4, -2e-4])
    plan.set_device(on, -2.7)
    T = plan.transmission(E, 1e-9)[0]
    assert plan.stats()["guard_redone"] == 4
    for e, tk in zip(E, T):
        assert abs(tk - closed_form_T(M, L, e)[0]) < 1e-9, (e, tk)
    # with disorder and a vacancy on either side of the junction slice m = L // 2 - 1
    on = inputs.anderson(M, L, 0.05, 5 + M)
    vac = np.zeros((L, M), dtype=np.uint8)
    m = L // 2 - 1
    vac[m, 2] = vac[m + 1, 5] = 1
    on[vac != 0] = inputs.VACANCY_ONSITE
    plan.set_device(on, -2.7, vac)
    E2 = np.array([4e-3, -4e-3, 2e-3])
    rgf.rgf_set_guard(plan.handle, 1e-14)          # force the pass for every energy
    T2 = plan.transmission(E2, 1e-9)[0]
    assert plan.stats()["guard_redone"] == 3
    rgf.rgf_set_guard(plan.handle, 1e-10)
    T_or = oracle.transmission_batch(on, vac, -2.7, E2, 1e-9)
    assert np.all(np.abs(T2 - T_or) <= tol(T_or)), np.abs(T2 - T_or)
