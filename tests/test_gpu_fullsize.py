"""Full-size parity: the configs of BASELINE.json in the launch configuration bench.py times
(whole energy batch in one rgf_transmission call), compared on the sampled energies whose oracle
value is stored under tests/golden/ (written by tests/golden/make_oracle_goldens.py, oracle only),
plus properties that hold at every energy.  Tolerance: |dT| <= 1e-9 * max(1, T)."""
import os

import numpy as np
import pytest

from paper_1107_5300_b200 import inputs

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def golden(cfg):
    g = np.loadtxt(os.path.join(GOLDEN, "config%d_oracle.txt" % cfg))
    return g[:, 0].astype(int), g[:, 1].astype(int), g[:, 2], g[:, 3]


def n_open_channels(M, E, t=-2.7):
    x = abs(E / t)
    return sum(1 for p in range(1, M // 2 + 1)
               if abs(1 - 2 * np.cos(p * np.pi / (M + 1))) < x < 1 + 2 * np.cos(p * np.pi / (M + 1)))


def check(w, T, cfg):
    dev, eidx, E, T_or = golden(cfg)
    assert np.allclose(w.energies[eidx], E, rtol=0, atol=0)
    got = T[dev, eidx]
    err = np.abs(got - T_or) / np.maximum(1.0, np.abs(T_or))
    assert np.all(err <= 1e-9), (cfg, err.max(), got, T_or)
    # properties at every energy (Q19): finite, 0 <= T <= number of open lead channels
    assert np.all(np.isfinite(T))
    nch = np.array([n_open_channels(w.M, e) for e in w.energies])
    assert np.all(T >= -1e-9) and np.all(T <= nch[None, :] + 1e-8), (T.min(), (T - nch[None, :]).max())
    return err.max()


@pytest.fixture()
def plan():
    from paper_1107_5300_b200 import binding as rgf
    with rgf.Plan(0) as p:
        yield p


def test_config1_four_seeds_batched(plan):
    w = inputs.config1()
    plan.set_device(w.onsite, w.t)
    T = plan.transmission(w.energies, w.eta)
    assert T.shape == (4, 256)
    check(w, T, 1)


def test_config2_headline(plan):
    w = inputs.config2()
    plan.set_device(w.onsite, w.t)
    T = plan.transmission(w.energies, w.eta)
    err = check(w, T, 2)
    st = plan.stats()
    print("configs[2]: max rel err %.2e, %.1f s, %d launches" % (err, st["ms_total"] / 1e3, st["launches"]))


def test_config3_disordered_c128(plan):
    w = inputs.config3(disordered=True)
    plan.set_device(w.onsite, w.t)
    T = plan.transmission(w.energies, w.eta)
    check(w, T, 3)


def test_config3_resonant_energies_against_80bit(plan):
    """configs[3], disordered, at energies inside the disorder band where the half-slice formulation alone is off by 2e-9 ... 4e-9
    (its singly bonded atoms are resonant at many slices) and the guard must hand the energy to the dense formulation: the
    default formulation, whole 1024-energy batch as bench-style runs launch it, against tests/golden/config3_ld.txt (80-bit
    arithmetic, written by tests/golden/make_near_neutrality_ld.py --config3: neither oracle nor CUDA)."""
    path = os.path.join(GOLDEN, "config3_ld.txt")
    rows = np.loadtxt(path, ndmin=2)
    idx, E, T_ld = rows[:, 0].astype(int), rows[:, 1], rows[:, 2]
    assert len(idx) >= 2
    w = inputs.config3(disordered=True)
    assert np.array_equal(w.energies[idx], E)
    plan.set_device(w.onsite, w.t)
    T = plan.transmission(w.energies, w.eta)[0]
    assert plan.stats()["guard_redone"] >= len(idx)
    err = np.abs(T[idx] - T_ld) / np.maximum(1.0, T_ld)
    assert np.all(err <= 1e-9), (err, T[idx], T_ld)


def test_config3_clean_c128_closed_form(plan):
    """configs[3] variant (a): clean M=244, L=2000 against the closed form (skip points within 1e-4 eV of a subband edge, Q8)."""
    from test_oracle_pins import closed_form_T
    w = inputs.config3(disordered=False)
    plan.set_device(w.onsite, w.t)
    T = plan.transmission(w.energies, w.eta)[0]
    skipped = 0
    for e, tk in zip(w.energies, T):
        Tc, n_open, dist = closed_form_T(w.M, w.L, e, eta=w.eta)
        if dist < 1e-4:
            skipped += 1
            continue
        assert abs(tk - Tc) < 1e-8 * max(1.0, Tc), (e, tk, Tc)
    assert skipped <= 16


def test_config4_wide_ribbon_truncated(plan):
    """configs[4] (M = 1024, edge vacancies): the first 64 slices of the same arrays, leads attached at slice 64, on 8
    energies (the naive oracle needs hours per energy at full length), element = each energy."""
    dev, eidx, E, T_or = golden(4)
    import re
    nsl = int(re.search(r"first (\d+) slices", open(os.path.join(GOLDEN, "config4_oracle.txt")).read()).group(1))
    assert nsl >= 24 and len(eidx) >= 4             # the golden's header names its truncation (64 slices x 8 energies once regenerated)
    w = inputs.truncate(inputs.config4(), nsl, eidx)
    assert np.array_equal(w.energies, E)
    plan.set_device(w.onsite, w.t, w.vacancy)
    T = plan.transmission(w.energies, w.eta)[0]
    err = np.abs(T - T_or) / np.maximum(1.0, np.abs(T_or))
    assert np.all(err <= 1e-9), (err.max(), T, T_or)


def lapack_referee_T(w, E):
    """Untimed LAPACK referee: the recursion of north_star written with torch-CPU inv / matmul (MKL), full M x M
    slices, batched over the energies E; leads by Sancho-Rubio in the M x M block form.  Test code only: it shares nothing
    with the CUDA path and is not the oracle (it is a library, so it referees where the naive oracle cannot reach)."""
    import torch
    M, L, t, eta = w.M, w.L, w.t, w.eta
    on = torch.from_numpy(w.onsite[0])
    vac = torch.from_numpy(w.vacancy[0].astype(bool)) if w.vacancy is not None else torch.zeros((L, M), dtype=torch.bool)
    nE = len(E)
    z = torch.tensor(E, dtype=torch.complex128) + 1j * eta
    eye = torch.eye(M, dtype=torch.complex128)
    j = torch.arange(M)

    def mask(i):
        return ((i + j) % 2 == 0).to(torch.float64)

    def H(i):            # slice Hamiltonian; i = None: clean lead slice
        h = torch.zeros((M, M), dtype=torch.complex128)
        alive = torch.ones(M - 1) if i is None else (~vac[i, :-1] & ~vac[i, 1:]).to(torch.float64)
        h[j[:-1], j[:-1] + 1] = t * alive.to(torch.complex128)
        h[j[:-1] + 1, j[:-1]] = t * alive.to(torch.complex128)
        if i is not None:
            h[j, j] = on[i].to(torch.complex128)
        return h

    def lead(pa, pb):    # surface Green's function of the lead cell (pa, pb): eliminate the second slice, decimate M x M blocks
        va, vb = t * mask(pa), t * mask(pb)
        G1 = torch.linalg.inv(z[:, None, None] * eye - H(None))
        eps_s = H(None) + va[:, None] * G1 * va[None, :]
        eps = eps_s + vb[:, None] * G1 * vb[None, :]
        al = va[:, None] * G1 * vb[None, :]
        be = al.transpose(1, 2).clone()
        for _ in range(64):
            if max(al.abs().max(), be.abs().max()) < 1e-14:
                break
            g = torch.linalg.inv(z[:, None, None] * eye - eps)
            agb, bga = al @ g @ be, be @ g @ al
            eps, eps_s = eps + agb + bga, eps_s + agb
            al, be = al @ g @ al, be @ g @ be
        return torch.linalg.inv(z[:, None, None] * eye - eps_s)

    gL = lead(-2, -1)
    gR = gL if L % 2 == 0 else lead(L, L + 1)
    mL = mask(-1) * (~vac[0]).to(torch.float64)
    mR = mask(L - 1) * (~vac[L - 1]).to(torch.float64)
    SigL = (t * mL)[:, None] * gL * (t * mL)[None, :]
    SigR = (t * mR)[:, None] * gR * (t * mR)[None, :]
    g = P = None
    for i in range(L):
        A = z[:, None, None] * eye - H(i)
        if i == 0:
            A = A - SigL
        else:
            m = t * mask(i - 1) * (~vac[i - 1]).to(torch.float64) * (~vac[i]).to(torch.float64)
            A = A - m[:, None] * g * m[None, :]
        if i == L - 1:
            A = A - SigR
        g = torch.linalg.inv(A)
        P = g[:, :, 1::2].clone() if i == 0 else (g * m[None, :]) @ P      # columns on which Gamma_L lives (odd j)
    GamL = (1j * (SigL - SigL.conj().transpose(1, 2)))[:, 1::2, 1::2]
    GamR = 1j * (SigR - SigR.conj().transpose(1, 2))
    Y = P.conj().transpose(1, 2) @ GamR @ P
    return torch.einsum("eab,eba->e", GamL, Y).real.numpy()


def test_lapack_referee_agrees_with_oracle(oracle):
    """The referee itself, pinned to the oracle where the oracle is quick (vacancies, odd L, disorder)."""
    w = inputs.truncate(inputs.config4(M=32, L=21, n_E=6), 21)
    T_ref = lapack_referee_T(w, w.energies)
    T_or = oracle.transmission_batch(w.onsite[0], w.vacancy[0], w.t, w.energies, w.eta)
    assert np.all(np.abs(T_ref - T_or) <= 1e-10 * np.maximum(1.0, T_or)), np.abs(T_ref - T_or)


@pytest.mark.parametrize("disordered", [False, True], ids=["clean", "disordered"])
def test_config3_c64_vs_c128(plan, disordered):
    """configs[3]: complex64 sweep against the complex128 sweep at all 1024 energies; north_star's bound is
    |dT| <= 1e-3 outside |E| < 0.1 eV (the growth towards charge neutrality is reported by precision_study.py)."""
    from paper_1107_5300_b200 import binding as rgf
    w = inputs.config3(disordered=disordered)
    plan.set_device(w.onsite, w.t)
    T128 = plan.transmission(w.energies, w.eta)[0]
    T64 = plan.transmission(w.energies, w.eta, precision=rgf.RGF_C64, ok=(rgf.RGF_ESINGULAR,))[0]
    outside = np.abs(w.energies) >= 0.1
    if not disordered:      # T(E) of the clean ribbon jumps at the subband edges: leave out energies within 1e-4 eV of one (Q8)
        from paper_1107_5300_b200.precision_study import edge_distance
        outside &= edge_distance(w.M, w.energies, w.t) >= 1e-4
        assert outside.sum() >= 400
    assert np.all(np.isfinite(T64[outside]))       # single precision may overflow only close to charge neutrality (reported)
    d = np.abs(np.where(np.isfinite(T64), T64, 0.0) - T128)
    assert d[outside].max() <= 1e-3, (d[outside].max(), w.energies[outside][np.argmax(d[outside])])      # north_star, literally
    assert d.max() > 1e-9          # a different precision really ran


def test_config4_wide_ribbon_full_length(plan):
    """configs[4] at full size (M = 1024, L = 2000, 64 energies, edge vacancies) in the launch configuration bench-style
    runs use.  No oracle value exists at this length (hours per energy with the naive LU), so: the properties that hold at
    any size on all 64 energies, and the LAPACK referee (lapack_referee_T, untimed, a few minutes of host time) at full
    length on 2 energies."""
    w = inputs.config4()
    plan.set_device(w.onsite, w.t, w.vacancy)
    T = plan.transmission(w.energies, w.eta)
    assert T.shape == (1, 64) and np.all(np.isfinite(T))
    nch = np.array([n_open_channels(w.M, e) for e in w.energies])
    assert np.all(T >= -1e-9) and np.all(T[0] <= nch + 1e-8), (T.min(), (T[0] - nch).max())
    st = plan.stats()
    print("configs[4] full length: %.1f s (leads %.1f s), %d launches" % (st["ms_total"] / 1e3, st["ms_leads"] / 1e3, st["launches"]))
    sub = np.array([5, 58])
    T_ref = lapack_referee_T(w, w.energies[sub])
    assert np.all(np.abs(T_ref - T[0, sub]) <= 1e-9 * np.maximum(1.0, T_ref)), (T_ref, T[0, sub])
