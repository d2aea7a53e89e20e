"""Pins of the CPU oracle to what the paper and the mathematics fix (no GPU, no CUDA library).

Each test cites the PAPER.md passage (line + equation) whose content it pins and is chosen so that a
plausible mistake in oracle/ref_lbm.cpp (a dropped term, a wrong sign or index, a transposed
operand, a wrong weight) fails at least one of them.  Nothing here calls paper_2502_12955_b200.
"""
import fractions
import os

import numpy as np
import pytest

import workloads
from oracle.ref_lbm import RefLBM, lattice_table

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def make(cfg):
    return RefLBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])


def rest_populations(w, rho):
    """f_i = w_i rho: the u = 0 equilibrium of Eq. 6; an input, not the method."""
    return np.stack([wi * rho for wi in w])


# ----------------------------------------------------------------------------------------------
# lattice tables: Tables 1-3
# ----------------------------------------------------------------------------------------------
def parse_golden():
    out, cur = {}, None
    for line in open(os.path.join(GOLDEN, "lattice_tables.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            cur = line.strip("[]")
            out[cur] = {}
            continue
        key, *vals = line.split()
        out[cur][key] = [float(fractions.Fraction(v)) for v in vals]
    return out


@pytest.mark.parametrize("name,lattice,kind", [("D3Q19", "D3Q19", 0), ("D2Q9", "D2Q9", 0), ("D2Q5", "D2Q9", 1)])
def test_lattice_tables_match_paper(name, lattice, kind):
    g = parse_golden()[name]
    c, w = lattice_table(lattice, kind)
    assert np.allclose(w, g["w"], rtol=0, atol=1e-16)
    assert np.array_equal(c[:, 0], np.array(g["cx"], int))
    assert np.array_equal(c[:, 1], np.array(g["cy"], int))
    if "cz" in g:
        assert np.array_equal(c[:, 2], np.array(g["cz"], int))
    else:
        assert not c[:, 2].any()


@pytest.mark.parametrize("lattice,kind,cs2", [("D3Q19", 0, 1 / 3), ("D2Q9", 0, 1 / 3), ("D2Q9", 1, 0.3), ("D3Q19", 1, 0.25)])
def test_lattice_isotropy(lattice, kind, cs2):
    """weights sum to one, sum w c = 0, sum w c_a c_b = c_s^2 delta_ab; every c has its opposite."""
    c, w = lattice_table(lattice, kind)
    d = 3 if lattice == "D3Q19" else 2
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs((w[:, None] * c).sum(0)).max() < 1e-16
    M = np.einsum("i,ia,ib->ab", w, c, c)[:d, :d]
    assert np.abs(M - cs2 * np.eye(d)).max() < 1e-15
    vecs = {tuple(v) for v in c.tolist()}
    assert len(vecs) == len(c) and all(tuple(-np.array(v)) in vecs for v in vecs)
    if kind == 0:  # fourth-order isotropy needed by Eq. 6: sum w c_a c_b c_g c_d = c_s^4 (dd + dd + dd)
        T = np.einsum("i,ia,ib,ic,id->abcd", w, c, c, c, c)[:d, :d, :d, :d]
        e = np.eye(d)
        iso = cs2 ** 2 * (np.einsum("ab,cd->abcd", e, e) + np.einsum("ac,bd->abcd", e, e) + np.einsum("ad,bc->abcd", e, e))
        assert np.abs(T - iso).max() < 1e-15


# ----------------------------------------------------------------------------------------------
# equilibrium, Eq. 6-8: moments of the initial (equilibrium) populations
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lattice,grid", [("D2Q9", (16, 12, 1)), ("D3Q19", (8, 8, 8))])
def test_equilibrium_moments(lattice, grid):
    r = RefLBM(*grid, lattice, "BGK", precision=64, tau=(0.8, 0.8), rho_init=(1.3, 1.0), u0=0.07, init_kind="TAYLOR_GREEN")
    r.init_from_seed(0)
    c, w = lattice_table(lattice)
    f, _ = r.split_populations(r.get_populations())
    f = f[0]
    m = r.get_macros()
    rho, u = m["rho"][0], m["u"]
    d = r.d
    assert np.abs(f.sum(0) - rho).max() < 1e-15
    for a in range(d):
        assert np.abs((c[:, a, None] * f).sum(0) - rho * u[a]).max() < 1e-16
    assert np.abs(u).max() > 0.05  # the velocity field is not trivially zero
    for a in range(d):
        for b in range(d):
            Pi = (c[:, a, None] * c[:, b, None] * f).sum(0)
            expect = rho * u[a] * u[b] + (rho / 3.0 if a == b else 0.0)
            assert np.abs(Pi - expect).max() < 1e-15


# ----------------------------------------------------------------------------------------------
# config 1: Taylor-Green decay, nu = (tau - 1/2)/3 ; pins BGK collision + periodic streaming
# Eq. 3-6
# ----------------------------------------------------------------------------------------------
def test_taylor_green_decay_cfg1():
    cfg = workloads.config("cfg1")
    r = make(cfg)
    r.init_from_seed(1)
    nx, ny, _ = cfg["grid"]
    k = 2 * np.pi / nx
    X, Y = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    mode_x = (-np.cos(k * X) * np.sin(k * Y)).ravel()
    mode_y = (np.sin(k * X) * np.cos(k * Y)).ravel()
    nu = (0.8 - 0.5) / 3.0
    amps, times = [], []
    mass0 = r.get_macros()["rho"].sum()
    t = 0
    for _ in range(10):
        r.step(100)
        t += 100
        m = r.get_macros()
        ax = (m["u"][0] * mode_x).sum() / (mode_x ** 2).sum()
        ay = (m["u"][1] * mode_y).sum() / (mode_y ** 2).sum()
        assert abs(ax - ay) < 1e-12  # the vortex stays symmetric
        # the field stays a pure mode
        assert np.abs(m["u"][0] - ax * mode_x).max() < 2e-4 * 0.01
        amps.append(ax)
        times.append(t)
    amps, times = np.array(amps), np.array(times)
    exact = 0.01 * np.exp(-2 * nu * k * k * times)
    assert abs(amps[-1] / exact[-1] - 1) < 5e-3          # amplitude at t = 1000 (0.145489 u0)
    rate = -np.polyfit(times[1:], np.log(amps[1:]), 1)[0]
    assert abs(rate / (2 * nu * k * k) - 1) < 1e-3       # decay rate pins nu = (tau-1/2)/3
    assert abs(r.get_macros()["rho"].sum() - mass0) < 1e-9


def test_taylor_green_viscosity_depends_on_tau():
    """the rate changes with tau as (tau - 1/2)/3: pins the 1/tau in Eq. 3 against e.g. tau vs 1/tau mix-ups"""
    rates = []
    for tau in (0.6, 1.0, 1.4):
        r = RefLBM(32, 32, 1, "D2Q9", "BGK", precision=64, tau=(tau, tau), u0=0.01, init_kind="TAYLOR_GREEN")
        r.init_from_seed(0)
        k = 2 * np.pi / 32
        X, Y = np.meshgrid(np.arange(32), np.arange(32), indexing="xy")
        mode = (-np.cos(k * X) * np.sin(k * Y)).ravel()
        r.step(100)
        a1 = (r.get_macros()["u"][0] * mode).sum() / (mode ** 2).sum()
        r.step(200)
        a2 = (r.get_macros()["u"][0] * mode).sum() / (mode ** 2).sum()
        rates.append(-np.log(a2 / a1) / 200 / (2 * k * k))
    assert np.allclose(rates, [(t - 0.5) / 3 for t in (0.6, 1.0, 1.4)], rtol=1.5e-2)


def test_taylor_green_3d_short_time():
    """Eq. 45 on D3Q19: at t -> 0 the kinetic energy decays at 2 nu |k|^2 with |k|^2 = 3 k^2."""
    n, tau = 24, 0.8
    r = RefLBM(n, n, n, "D3Q19", "BGK", precision=64, tau=(tau, tau), u0=0.002, init_kind="TAYLOR_GREEN")
    r.init_from_seed(0)
    k = 2 * np.pi / n

    def energy():
        m = r.get_macros()
        return float((m["u"] ** 2).sum())

    r.step(20)
    e1 = energy()
    r.step(40)
    e2 = energy()
    rate = -np.log(e2 / e1) / 40
    nu = (tau - 0.5) / 3
    assert abs(rate / (2 * nu * 3 * k * k * 2 / 2) - 1) < 0.02  # energy ~ amplitude^2: 2 * (nu * 3 k^2)


# ----------------------------------------------------------------------------------------------
# config 4: Guo body force + halfway bounce-back walls -> Poiseuille parabola (PAPER.md:504-531,
# Eq. 43-44 with the missing 1/2 restored; Eq. 20-23; bounce-back PAPER.md:446, 525)
# ----------------------------------------------------------------------------------------------
def poiseuille_exact(nz, tau, g):
    nu = (tau - 0.5) / 3
    z = np.arange(nz)
    return (g / (2 * nu)) * (z + 0.5) * (nz - z - 0.5) + (g / (8 * nu)) * (16 * (tau - 0.5) ** 2 / 3 - 1)


@pytest.mark.parametrize("tau", [0.6, 0.9, 0.5 + np.sqrt(3.0 / 16.0), 1.2])
def test_poiseuille_profile(tau):
    nz, g = 16, 1e-6
    cfg = workloads.config("cfg4", grid=(1, 1, nz), tau=(tau, tau))
    r = make(cfg)
    r.init_from_seed(0)
    r.step(int(30 * nz * nz / ((tau - 0.5) / 3)))
    m = r.get_macros()
    ex = poiseuille_exact(nz, tau, g)
    assert np.abs(m["u"][0] - ex).max() / ex.max() < 1e-8
    assert np.abs(m["u"][1]).max() == 0 and np.abs(m["u"][2]).max() < 1e-12   # round-off only
    assert np.abs(m["rho"] - 1).max() < 1e-10                 # round-off accumulated over ~1e5 steps
    # discrete second difference = -g/nu exactly (independent of the wall slip)
    d2 = m["u"][0][2:] - 2 * m["u"][0][1:-1] + m["u"][0][:-2]
    assert np.allclose(d2, -g / ((tau - 0.5) / 3), rtol=1e-6)


def test_poiseuille_xy_invariance_is_bit_exact():
    """a 3x2xnz channel equals the 1x1xnz one bit for bit (used by the 256^3 GPU parity test)"""
    nz = 12
    a = make(workloads.config("cfg4", grid=(1, 1, nz)))
    b = make(workloads.config("cfg4", grid=(3, 2, nz)))
    for r in (a, b):
        r.init_from_seed(0)
        r.step(57)
    ua, ub = a.get_macros()["u"], b.get_macros()["u"].reshape(3, nz, 2, 3)
    for x in range(3):
        for y in range(2):
            assert np.array_equal(ub[:, :, y, x], ua)
    fa = a.get_populations().reshape(19, nz)
    fb = b.get_populations().reshape(19, nz, 6)
    assert np.array_equal(fb[:, :, 4], fa)


def test_walls_on_other_axes_and_2d():
    """the same channel with walls on x (3D) and on y (2D): pins the bounce-back index logic per axis"""
    n, tau, g = 12, 0.9, 1e-6
    ex = poiseuille_exact(n, tau, g)
    r = RefLBM(n, 1, 1, "D3Q19", "BGK", precision=64, tau=(tau, tau), force=(0, g, 0), bc=(1, 0, 0))
    r.init_from_seed(0)
    r.step(40000)
    assert np.abs(r.get_macros()["u"][1] - ex).max() / ex.max() < 1e-8
    r = RefLBM(1, n, 1, "D2Q9", "BGK", precision=64, tau=(tau, tau), force=(g, 0, 0), bc=(0, 1, 0))
    r.init_from_seed(0)
    r.step(40000)
    assert np.abs(r.get_macros()["u"][0] - ex).max() / ex.max() < 1e-8


def test_poiseuille_fp32_close_to_closed_form():
    nz, tau, g = 16, 0.9, 1e-5
    r = make(workloads.config("cfg4", grid=(1, 1, nz), precision=32, force=(g, 0, 0)))
    r.init_from_seed(0)
    r.step(60000)
    ex = poiseuille_exact(nz, tau, g)
    assert np.abs(r.get_macros()["u"][0] - ex).max() / ex.max() < 2e-3


# ----------------------------------------------------------------------------------------------
# Guo forcing bookkeeping, Eq. 15, 20, 22
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lattice,grid,force", [("D2Q9", (6, 5, 1), (3e-5, -2e-5, 0.0)), ("D3Q19", (4, 5, 3), (1e-5, 2e-5, -3e-5))])
def test_uniform_force_momentum_growth(lattice, grid, force):
    """periodic box, uniform force density F: every step adds exactly F to the momentum of each cell, and the
    physical velocity carries the half-force shift: u(t) = F (t + 1/2) / rho.  Pins (1 - 1/2tau) F_i and F/2."""
    tau = 0.77
    r = RefLBM(*grid, lattice, "BGK", precision=64, tau=(tau, tau), force=force, rho_init=(1.25, 1.0))
    r.init_from_seed(0)
    c, _ = lattice_table(lattice)
    for t in (0, 1, 7, 40):
        if t:
            r.step(t - r_t)
        r_t = t
        m = r.get_macros()
        f, _ = r.split_populations(r.get_populations())
        for a in range(r.d):
            assert np.allclose(m["u"][a], force[a] * (t + 0.5) / 1.25, rtol=1e-11, atol=1e-19)
            mom = (c[:, a, None] * f[0]).sum(0)
            assert np.allclose(mom, force[a] * t, rtol=1e-10, atol=1e-18)
        assert np.abs(m["rho"] - 1.25).max() < 1e-13


def noise_cfg(model, lattice, grid, precision=64, **kw):
    base = dict(precision=precision, tau=(1.0, 0.9), tau_c=0.8, psi_kind=1, G=workloads.G12, k_react=0.0,
                init_kind="UNIFORM_NOISE", rho_init=(1.0, 0.8), noise_amp=0.05, c_init=0.7)
    if model == "SC1":
        base.update(psi_kind=0, G=((-5.0, 0), (0, 0)), rho_init=(0.7, 1.0))
    base.update(kw)
    return RefLBM(*grid, lattice, model, **base)


@pytest.mark.parametrize("model,lattice,grid", [
    ("BGK", "D2Q9", (9, 7, 1)), ("SC1", "D2Q9", (16, 16, 1)), ("SC2", "D2Q9", (16, 12, 1)), ("SC2_ADE", "D2Q9", (12, 12, 1)),
    ("SC1", "D3Q19", (8, 6, 7)), ("SC2_ADE", "D3Q19", (8, 8, 6))])
def test_mass_and_momentum_conservation(model, lattice, grid):
    """sum_x rho^sigma is invariant (sum_i F_i = 0, sum_i f^eq = rho); the Shan-Chen force sums to zero over a
    periodic box, so the total momentum sum_x sum_sigma j^sigma is invariant too; k = 0 conserves sum C."""
    # total momentum is conserved by the multi-component Guo scheme only for equal relaxation times:
    # sum_sigma omega^sigma (j^sigma - rho^sigma u^b) = -omega sum F / 2 needs a common omega (Eq. 15, 20)
    r = noise_cfg(model, lattice, grid, tau=(0.9, 0.9))
    r.init_from_seed(11)
    c, _ = lattice_table(lattice)

    def totals():
        f, h = r.split_populations(r.get_populations())
        mass = f.sum(axis=(1, 2))
        mom = np.array([(c[:, a, None] * f.sum(0)).sum() for a in range(r.d)])
        return mass, mom, (h.sum() if h is not None else 0.0)

    m0, p0, c0 = totals()
    r.step(200)
    m1, p1, c1 = totals()
    assert np.abs(m1 - m0).max() / m0.max() < 1e-13
    assert np.abs(p1 - p0).max() / m0.sum() < 1e-13
    assert abs(c1 - c0) <= 1e-13 * max(abs(c0), 1)
    if model != "BGK":
        F = r.get_force()
        assert np.abs(F.sum(axis=(0, 2))).max() < 1e-12          # Newton's third law over the box
        assert np.abs(F).max() > 1e-5                            # ... of a force that is not trivially zero


# ----------------------------------------------------------------------------------------------
# Shan-Chen force against the literal pair sum of Eq. 9, discretised as stated
# at PAPER.md:126: G(x~ - x) = w_i G if x~ - x = c_i, else 0.   Eq. 11 / 13
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("model,lattice,grid", [("SC1", "D2Q9", (8, 8, 1)), ("SC2", "D2Q9", (8, 8, 1)), ("SC2_ADE", "D3Q19", (6, 6, 6))])
def test_shan_chen_force_equals_pair_sum(model, lattice, grid):
    G = ((-5.0, 0.0), (0.0, 0.0)) if model == "SC1" else ((0.3, 1.2), (1.2, -0.4))
    r = noise_cfg(model, lattice, grid, G=G)
    r.init_from_seed(5)
    r.step(3)  # a state with non-trivial velocity
    m = r.get_macros()
    F = r.get_force()
    nx, ny, nz = grid
    c, w = lattice_table(lattice)
    S, d, N = r.S, r.d, r.N
    rho = m["rho"]
    psi = rho if model != "SC1" else 1.0 - np.exp(-rho)
    wmap = {tuple(ci): wi for ci, wi in zip(c.tolist(), w)}
    coords = [(x, y, z) for z in range(nz) for y in range(ny) for x in range(nx)]
    Fb = np.zeros((S, d, N))
    for a_idx, xa in enumerate(coords):
        for b_idx, xb in enumerate(coords):
            if a_idx == b_idx:
                continue
            # every periodic image of xb that is a lattice neighbour of xa
            for sx in (-nx, 0, nx):
                for sy in (-ny, 0, ny):
                    for sz in ((-nz, 0, nz) if nz > 1 else (0,)):
                        dv = (xb[0] + sx - xa[0], xb[1] + sy - xa[1], xb[2] + sz - xa[2])
                        wi = wmap.get(dv)
                        if wi is None:
                            continue
                        for s in range(S):
                            for t in range(S):
                                for a in range(d):
                                    Fb[s, a, a_idx] -= dv[a] * wi * G[s][t] * psi[s, a_idx] * psi[t, b_idx]
    assert np.abs(F - Fb).max() < 1e-14
    assert np.abs(Fb).max() > 1e-3


def test_shan_chen_force_uniform_and_linear_psi():
    """uniform psi -> F = 0; psi linear in x -> F_x = -G psi c_s^2 dpsi/dx (continuum limit of Eq. 11)"""
    nx, ny = 16, 6
    c, w = lattice_table("D2Q9")
    r = RefLBM(nx, ny, 1, "D2Q9", "SC1", precision=64, tau=(1, 1), psi_kind=1, G=((-3.0, 0), (0, 0)))
    x = np.arange(nx)
    for slope in (0.0, 0.01):
        rho = np.tile(1.0 + slope * x, ny)
        r.set_populations(rest_populations(w, rho).ravel())
        F = r.get_force()[0].reshape(2, ny, nx)
        inner = slice(1, nx - 1)
        expect = -(-3.0) * (1.0 + slope * x[inner]) * (1.0 / 3.0) * slope
        assert np.abs(F[0][:, inner] - expect).max() < 1e-15
        assert np.abs(F[1][:, inner]).max() < 1e-16


def test_shan_chen_3d_gradient_each_axis():
    c, w = lattice_table("D3Q19")
    n = 8
    r = RefLBM(n, n, n, "D3Q19", "SC1", precision=64, tau=(1, 1), psi_kind=1, G=((2.0, 0), (0, 0)))
    idx = np.indices((n, n, n))  # [z, y, x] order of axes -> map axis a to array
    for a in range(3):
        coord = idx[2 - a].ravel().astype(float)
        rho = 1.0 + 0.02 * coord
        r.set_populations(rest_populations(w, rho).ravel())
        F = r.get_force()[0]
        inner = (coord > 0) & (coord < n - 1)
        for b in range(3):
            expect = -2.0 * rho * (1 / 3) * 0.02 if a == b else 0.0 * rho
            assert np.abs((F[b] - expect)[inner]).max() < 1e-15


# ----------------------------------------------------------------------------------------------
# config 2: Laplace law, Eq. 47, with the single-component EOS p = rho/3 + G psi^2/6
# ----------------------------------------------------------------------------------------------
@pytest.mark.slow
def test_laplace_law_reduced_cfg2():
    n = 96
    res = []
    for R in (12, 17, 22):
        cfg = workloads.config("cfg2", grid=(n, n, 1), radius=float(R))
        r = make(cfg)
        r.init_from_seed(7)
        mass0 = r.get_macros()["rho"].sum()
        r.step(5000)
        m = r.get_macros()
        rho = m["rho"][0].reshape(n, n)
        assert abs(rho.sum() - mass0) / mass0 < 1e-11           # mass conservation
        psi = 1 - np.exp(-rho)
        p = rho / 3 + (-5.0 / 6) * psi ** 2
        rin, rout = rho[n // 2, n // 2], rho[0, 0]
        assert rin > 1.8 and rout < 0.2                          # liquid inside, vapour outside
        reff = np.sqrt(((rho - rout) / (rin - rout)).sum() / np.pi)
        res.append((1 / reff, p[n // 2, n // 2] - p[0, 0]))
        assert np.abs(m["u"]).max() < 0.02                       # spurious currents stay small
    inv_r, dp = np.array(res).T
    gamma = dp / inv_r
    assert (dp > 0).all() and (np.diff(dp) < 0).all()            # larger droplet, smaller jump
    assert gamma.max() / gamma.min() - 1 < 0.05                  # dp * R constant
    slope = (inv_r * dp).sum() / (inv_r ** 2).sum()              # line through the origin
    assert np.abs(dp - slope * inv_r).max() / dp.max() < 0.03


# ----------------------------------------------------------------------------------------------
# two components: EOS Eq. 46 and the critical coupling G_c > 1/(rho1+rho2)...
# ----------------------------------------------------------------------------------------------
def test_two_component_flat_interface_pressure_balance():
    """an asymmetric A-rich / B-rich slab relaxes until P = (rhoA+rhoB)/3 + G12 rhoA rhoB / 3 is equal in both
    bulks although the ideal part (rhoA+rhoB)/3 differs by several per cent: pins the magnitude of Eq. 13."""
    nx, ny = 2, 128
    _, w = lattice_table("D2Q9")
    y = np.arange(ny)
    I = 0.5 * (1 + np.tanh((y - 32) / 2.0)) * 0.5 * (1 - np.tanh((y - 96) / 2.0))
    rA, rB = np.repeat(0.05 + 1.85 * I, nx), np.repeat(1.4 - 1.35 * I, nx)
    r = RefLBM(nx, ny, 1, "D2Q9", "SC2", precision=64, tau=(1.0, 1.0), psi_kind=1, G=workloads.G12)
    r.set_populations(np.concatenate([rest_populations(w, rA).ravel(), rest_populations(w, rB).ravel()]))
    r.step(15000)
    rho = r.get_macros()["rho"].reshape(2, ny, nx)[:, :, 0]
    P = (rho[0] + rho[1]) / 3 + 1.2 * rho[0] * rho[1] / 3
    ideal = (rho[0] + rho[1]) / 3
    assert abs(P[64] - P[0]) / P[0] < 1e-3
    assert abs(ideal[64] - ideal[0]) / ideal[0] > 0.03
    assert rho[0, 64] > 1.2 and rho[1, 0] > 1.0                  # still demixed


def test_two_component_demixing_threshold():
    """psi = rho, rhoA = rhoB = 1: noise grows iff G12 sqrt(rhoA rhoB) > 1 (config 3 is above it; reading R3)"""
    out = {}
    for G12 in (0.8, 1.2):
        cfg = workloads.config("cfg3", grid=(48, 48, 1), G=((0, G12), (G12, 0)))
        r = make(cfg)
        r.init_from_seed(3)
        d0 = np.abs(np.diff(r.get_macros()["rho"], axis=0)).max()
        r.step(600)
        out[G12] = np.abs(np.diff(r.get_macros()["rho"], axis=0)).max() / d0
    assert out[0.8] < 0.5 and out[1.2] > 5.0


# ----------------------------------------------------------------------------------------------
# scalar lattice, Eq. 34-36: diffusion, advection, first-order source
# ----------------------------------------------------------------------------------------------
def scalar_setup(lattice, grid, u, Cfield, rhoA=1.0, rhoB=1.0, **kw):
    """SC2_ADE context with G = 0 (the flow is a uniform fixed point) moving at velocity u; inputs are built from
    the lattice tables only."""
    c, w = lattice_table(lattice, 0)
    cs, ws = lattice_table(lattice, 1)
    d = 3 if lattice == "D3Q19" else 2
    cs2g = (1 - ws[0]) / d
    par = dict(precision=64, tau=(1.0, 1.0), tau_c=0.8, psi_kind=1, G=((0, 0), (0, 0)), k_react=0.0)
    par.update(kw)
    r = RefLBM(*grid, lattice, "SC2_ADE", **par)
    N = r.N
    u = np.asarray(u, float)
    cu = c[:, :d] @ u[:d]
    feq = w * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * (u[:d] @ u[:d]))
    fA = np.outer(feq, np.full(N, rhoA))
    fB = np.outer(feq, np.full(N, rhoB))
    heq = ws[:, None] * Cfield[None, :] * (1 + (cs[:, :d] @ u[:d])[:, None] / cs2g)
    r.set_populations(np.concatenate([fA.ravel(), fB.ravel(), heq.ravel()]))
    return r


@pytest.mark.parametrize("lattice,grid,axis", [("D2Q9", (64, 2, 1), 0), ("D2Q9", (2, 64, 1), 1),
                                               ("D3Q19", (64, 2, 2), 0), ("D3Q19", (2, 64, 2), 1), ("D3Q19", (2, 2, 64), 2)])
def test_scalar_diffusion_and_advection(lattice, grid, axis):
    """a sine mode of C decays as exp(-D k^2 t), D = c_sg^2 (tau_c - 1/2) [tau_d = D/c_sg^2 + 1/2 is the paper's
    (10/3) D + 0.5 for D2Q5, PAPER.md:336] and translates at the fluid velocity u (Eq. 35)."""
    d = 3 if lattice == "D3Q19" else 2
    n = 64
    idx = np.indices(grid[::-1])[2 - axis].ravel().astype(float)  # coordinate along `axis` per cell
    k = 2 * np.pi / n
    cs2g = 0.3 if d == 2 else 0.25
    D = cs2g * (0.8 - 0.5)
    for speed in (0.0, 0.05):
        u = np.zeros(3)
        u[axis] = speed
        r = scalar_setup(lattice, grid, u, 1.0 + 0.1 * np.sin(k * idx))
        T = 400
        r.step(T)
        m = r.get_macros()
        C = m["C"]
        assert np.allclose(m["u"][axis], speed, atol=1e-14)
        a_s = 2 * ((C - 1) * np.sin(k * idx)).mean()
        a_c = 2 * ((C - 1) * np.cos(k * idx)).mean()
        amp = np.hypot(a_s, a_c)
        # second-order advection correction of the LBGK scheme: D_eff = D - (tau_c - 1/2) u^2
        d_eff = D - (0.8 - 0.5) * speed ** 2
        assert abs(amp / (0.1 * np.exp(-d_eff * k * k * T)) - 1) < 3e-3
        shift = np.arctan2(-a_c, a_s) / k
        assert abs(shift - speed * T) < 0.02
        assert abs(C.mean() - 1) < 1e-13                          # k_react = 0 conserves sum C


@pytest.mark.parametrize("lattice,grid", [("D2Q9", (5, 4, 1)), ("D3Q19", (4, 3, 5))])
def test_scalar_first_order_reaction_uniform_state(lattice, grid):
    """uniform state: C(t) = C0 (1 - k chi)^t exactly, chi = 4 rhoA rhoB / (rhoA + rhoB)^2 (BASELINE.json config 5)"""
    N = int(np.prod(grid))
    kr, rA, rB, C0 = 1e-3, 1.5, 0.5, 0.8
    r = scalar_setup(lattice, grid, (0, 0, 0), np.full(N, C0), rhoA=rA, rhoB=rB, k_react=kr)
    chi = 4 * rA * rB / (rA + rB) ** 2
    for T in (1, 10, 300):
        r.step(T if T == 1 else (9 if T == 10 else 290))
        C = r.get_macros()["C"]
        assert np.abs(C / (C0 * (1 - kr * chi) ** T) - 1).max() < 1e-13
    # a pure component (chi = 0) does not react
    r = scalar_setup(lattice, grid, (0, 0, 0), np.full(N, C0), rhoA=1.0, rhoB=0.0, k_react=kr)
    r.step(50)
    assert np.abs(r.get_macros()["C"] - C0).max() < 1e-15


# ----------------------------------------------------------------------------------------------
# fixed points and symmetry
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("model,lattice,grid", [("BGK", "D2Q9", (5, 4, 1)), ("SC1", "D2Q9", (5, 4, 1)),
                                                ("SC2_ADE", "D2Q9", (5, 4, 1)), ("SC2_ADE", "D3Q19", (4, 3, 3))])
def test_uniform_rest_state_is_stationary(model, lattice, grid):
    r = noise_cfg(model, lattice, grid, noise_amp=0.0, init_kind="REST", k_react=0.0)
    r.init_from_seed(0)
    f0 = r.get_populations()
    r.step(25)
    assert np.abs(r.get_populations() - f0).max() < 1e-15
    assert np.abs(r.get_macros()["u"]).max() < 1e-16


def rotation_maps(lattice, grid):
    """90-degree rotation about z: (x, y) -> (-y, x).  Returns the rotated grid, the cell map and the
    direction permutations of the flow and scalar lattices (built from the tables)."""
    nx, ny, nz = grid
    gx, gy = ny, nx
    cell_map = np.empty(nx * ny * nz, int)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                xr, yr = (gx - 1 - y), x
                cell_map[x + nx * (y + ny * z)] = xr + gx * (yr + gy * z)
    perms = []
    for kind in (0, 1):
        c, _ = lattice_table(lattice, kind)
        lut = {tuple(v): i for i, v in enumerate(c.tolist())}
        perms.append(np.array([lut[(-v[1], v[0], v[2])] for v in c.tolist()]))
    return (gx, gy, nz), cell_map, perms


@pytest.mark.parametrize("model,lattice,grid", [("SC2_ADE", "D2Q9", (8, 6, 1)), ("SC1", "D2Q9", (7, 5, 1)), ("SC2_ADE", "D3Q19", (6, 4, 5))])
def test_rotation_equivariance(model, lattice, grid):
    """rotating the input by 90 degrees (cells and lattice directions) rotates the output: catches any
    inconsistency between the velocity table, the streaming offsets and the force / equilibrium terms."""
    a = noise_cfg(model, lattice, grid, k_react=1e-3, force=(0.0, 0.0, 0.0))
    a.init_from_seed(9)
    a.step(2)
    fa, ha = a.split_populations(a.get_populations())
    g2, cmap, (pf, ph) = rotation_maps(lattice, grid)
    b = noise_cfg(model, lattice, g2, k_react=1e-3)
    fb = np.empty_like(fa)
    fb[:, pf[:, None], cmap[None, :]] = fa
    parts = [fb.ravel()]
    if ha is not None:
        hb = np.empty_like(ha)
        hb[ph[:, None], cmap[None, :]] = ha
        parts.append(hb.ravel())
    b.set_populations(np.concatenate(parts))
    a.step(20)
    b.step(20)
    fa2, ha2 = a.split_populations(a.get_populations())
    fb2, hb2 = b.split_populations(b.get_populations())
    assert np.abs(fb2[:, pf[:, None], cmap[None, :]] - fa2).max() < 1e-14
    if ha2 is not None:
        assert np.abs(hb2[ph[:, None], cmap[None, :]] - ha2).max() < 1e-14
    assert np.abs(fa2 - fa).max() > 1e-4                         # the state did evolve


def test_streaming_moves_each_population_along_its_velocity():
    """tau = 1 and u = 0 equilibrium everywhere except one marked population: after one step the excess of f_i
    sits at x + c_i (Eq. 5); pins the direction table against the streaming offsets."""
    for lattice, grid in (("D2Q9", (5, 6, 1)), ("D3Q19", (5, 6, 4))):
        c, w = lattice_table(lattice)
        nx, ny, nz = grid
        N = nx * ny * nz
        for i in range(len(w)):
            r = RefLBM(*grid, lattice, "BGK", precision=64, tau=(1e9, 1e9))  # omega ~ 0: no relaxation
            f = rest_populations(w, np.ones(N))
            x0 = (2, 3, 1 if nz > 1 else 0)
            cell0 = x0[0] + nx * (x0[1] + ny * x0[2])
            f[i, cell0] += 0.5
            r.set_populations(f.ravel())
            r.step(1)
            f1, _ = r.split_populations(r.get_populations())
            x1 = ((x0[0] + c[i, 0]) % nx, (x0[1] + c[i, 1]) % ny, (x0[2] + c[i, 2]) % nz)
            cell1 = x1[0] + nx * (x1[1] + ny * x1[2])
            excess = f1[0] - rest_populations(w, np.ones(N))
            assert abs(excess[i, cell1] - 0.5) < 1e-9
            excess[i, cell1] = 0
            assert np.abs(excess).max() < 1e-9


def test_bounce_back_reverses_population_at_wall():
    """halfway bounce-back: a population leaving through a wall is back in the same cell, in the
    opposite direction, at t + 1; wall-parallel motion and the periodic axes are untouched."""
    c, w = lattice_table("D3Q19")
    nx, ny, nz = 4, 3, 4
    N = nx * ny * nz
    for i in range(19):
        r = RefLBM(nx, ny, nz, "D3Q19", "BGK", precision=64, tau=(1e9, 1e9), bc=(0, 0, 1))
        f = rest_populations(w, np.ones(N))
        x0 = (1, 1, 0)  # bottom layer
        cell0 = x0[0] + nx * (x0[1] + ny * x0[2])
        f[i, cell0] += 0.5
        r.set_populations(f.ravel())
        r.step(1)
        f1, _ = r.split_populations(r.get_populations())
        excess = f1[0] - rest_populations(w, np.ones(N))
        if c[i, 2] < 0:
            opp = [j for j in range(19) if (c[j] == -c[i]).all()][0]
            assert abs(excess[opp, cell0] - 0.5) < 1e-9
        else:
            x1 = ((x0[0] + c[i, 0]) % nx, (x0[1] + c[i, 1]) % ny, x0[2] + c[i, 2])
            assert abs(excess[i, x1[0] + nx * (x1[1] + ny * x1[2])] - 0.5) < 1e-9
        assert abs(excess.sum() - 0.5) < 1e-9


# ----------------------------------------------------------------------------------------------
# precision variants and the seeded inputs
# ----------------------------------------------------------------------------------------------
def test_fp32_oracle_tracks_fp64_oracle():
    a = noise_cfg("SC2_ADE", "D3Q19", (8, 8, 8), precision=64, k_react=1e-3)
    b = noise_cfg("SC2_ADE", "D3Q19", (8, 8, 8), precision=32, k_react=1e-3)
    for r in (a, b):
        r.init_from_seed(4)
        r.step(50)
    ma, mb = a.get_macros(), b.get_macros()
    assert mb["rho"].dtype == np.float32
    for key in ("rho", "C"):
        assert np.abs(ma[key] - mb[key]).max() / np.abs(ma[key]).max() < 2e-6
    assert np.abs(ma["u"] - mb["u"]).max() < 1e-6


def test_seeded_noise_statistics_and_reproducibility():
    cfg = workloads.config("cfg3", grid=(64, 64, 1))
    a, b, c3 = make(cfg), make(cfg), make(cfg)
    a.init_from_seed(1)
    b.init_from_seed(1)
    c3.init_from_seed(2)
    ra, rb, rc = (r.get_macros()["rho"] for r in (a, b, c3))
    assert np.array_equal(ra, rb) and not np.array_equal(ra, rc)
    dev = (ra - 1.0) / 0.01                                          # uniform in [-1, 1)
    assert dev.min() >= -1 - 1e-12 and dev.max() < 1 + 1e-12
    assert abs(dev.mean()) < 0.03 and abs(dev.std() - 1 / np.sqrt(3)) < 0.02
    assert abs(np.corrcoef(ra[0], ra[1])[0, 1]) < 0.05             # components use different streams


def test_random_droplets_volume_fraction():
    cfg = workloads.config("cfg5", grid=(64, 64, 64), rmin=5.0, rmax=10.0)
    r = make(cfg)
    r.init_from_seed(12)
    m = r.get_macros()
    rhoA, rhoB, Cc = m["rho"][0], m["rho"][1], m["C"]
    assert abs(rhoA.min() - 0.1) < 1e-6 and abs(rhoA.max() - 1.9) < 1e-6
    assert np.abs(rhoA + rhoB - 2.0).max() < 1e-6                   # total density 2 everywhere
    frac = (Cc > 0.5).mean()
    assert 0.03 < frac < 0.09                                       # about the 5 % requested (overlaps allowed)
    assert np.abs(Cc - (rhoA - 0.1) / 1.8).max() < 1e-6             # C = 1 inside A, 0 outside


def test_errors():
    with pytest.raises(ValueError):
        RefLBM(4, 4, 2, "D2Q9", "BGK")                             # 2D lattice with nz != 1
    with pytest.raises(ValueError):
        RefLBM(4, 4, 1, "D2Q9", "BGK", tau=(0.5, 1.0))
    with pytest.raises(ValueError):
        RefLBM(4, 4, 1, "D2Q9", "BGK", forcing=2)
    r = RefLBM(4, 4, 1, "D2Q9", "BGK")
    with pytest.raises(RuntimeError):
        r.step(1)                                                    # step before init


# ----------------------------------------------------------------------------------------------
# Shan-Chen (velocity-shift) forcing scheme, forcing = 1: Eq. 16-19
# ----------------------------------------------------------------------------------------------
def test_velocity_shift_without_force_is_plain_bgk():
    """F = 0: u^eq = u' = j / rho (Eq. 16-17 with one component), so the scheme is the LBGK update itself."""
    kw = dict(precision=64, tau=(0.8, 0.8), init_kind="TAYLOR_GREEN", u0=0.03, rho_init=(1.1, 1.0))
    a = RefLBM(12, 10, 1, "D2Q9", "BGK", forcing=0, **kw)
    b = RefLBM(12, 10, 1, "D2Q9", "BGK", forcing=1, **kw)
    a.init_from_seed(0); b.init_from_seed(0)
    a.step(60); b.step(60)
    fa, fb = a.get_populations(), b.get_populations()
    assert np.abs(fa - fb).max() <= 1e-14 * np.abs(fa).max()


@pytest.mark.parametrize("lattice,grid,force", [("D2Q9", (6, 5, 1), (3e-5, -2e-5, 0.0)), ("D3Q19", (4, 5, 3), (1e-5, 2e-5, -3e-5))])
def test_velocity_shift_uniform_force_momentum_growth(lattice, grid, force):
    """The first moment of f^eq(rho, u' + tau F / rho) is j + tau F, so relaxing towards it adds exactly F to
    the momentum of each cell per step (Eq. 15-16); the physical velocity carries F/2 (Eq. 19)."""
    tau = 0.77
    r = RefLBM(*grid, lattice, "BGK", precision=64, tau=(tau, tau), force=force, rho_init=(1.25, 1.0), forcing=1)
    r.init_from_seed(0)
    c, _ = lattice_table(lattice)
    done = 0
    for t in (0, 1, 7, 40):
        r.step(t - done); done = t
        m = r.get_macros()
        f, _ = r.split_populations(r.get_populations())
        for a in range(r.d):
            assert np.allclose(m["u"][a], force[a] * (t + 0.5) / 1.25, rtol=1e-11, atol=1e-19)
            assert np.allclose((c[:, a, None] * f[0]).sum(0), force[a] * t, rtol=1e-10, atol=1e-18)
        assert np.abs(m["rho"] - 1.25).max() < 1e-13


@pytest.mark.parametrize("model,lattice,grid", [("SC2", "D2Q9", (16, 12, 1)), ("SC2_ADE", "D3Q19", (8, 8, 6)), ("SC1", "D2Q9", (16, 16, 1))])
def test_velocity_shift_conserves_momentum_with_unequal_relaxation_times(model, lattice, grid):
    """With u' weighted by rho^s / tau^s (Eq. 17) the relaxation terms of the components cancel in the sum:
    sum_s (j^s - rho^s u') / tau^s = 0, so the total momentum of a periodic box changes by sum F = 0 only --
    for ANY tau^A != tau^B (a plain average in Eq. 17 would break this).  Mass per component is invariant."""
    r = noise_cfg(model, lattice, grid, tau=(1.0, 0.7), forcing=1)
    r.init_from_seed(5)
    c, _ = lattice_table(lattice)

    def totals():
        f, _ = r.split_populations(r.get_populations())
        return f.sum(axis=(1, 2)), np.array([(c[:, a, None] * f.sum(0)).sum() for a in range(r.d)])

    m0, p0 = totals()
    r.step(150)
    m1, p1 = totals()
    assert np.abs(m1 - m0).max() / m0.max() < 1e-13
    assert np.abs(p1 - p0).max() / m0.sum() < 1e-13
    assert np.abs(r.get_force()).max() > 1e-5


def test_velocity_shift_poiseuille_curvature():
    """Body force + halfway bounce-back walls under the velocity-shift scheme: the steady profile is a parabola
    of curvature -g / nu with nu = (tau - 1/2) / 3 (the extra tau^2 F F / rho momentum flux of this scheme is
    uniform here), symmetric about the channel centre."""
    nz, g, tau = 16, 1e-6, 0.9
    cfg = workloads.config("cfg4", grid=(1, 1, nz), tau=(tau, tau), forcing=1)
    r = make(cfg)
    r.init_from_seed(0)
    nu = (tau - 0.5) / 3
    r.step(int(30 * nz * nz / nu))
    u = r.get_macros()["u"][0]
    d2 = u[2:] - 2 * u[1:-1] + u[:-2]
    assert np.allclose(d2, -g / nu, rtol=1e-6)
    assert np.allclose(u, u[::-1], rtol=1e-9)
    assert u.max() > 0.9 * g * nz * nz / (8 * nu)


def test_velocity_shift_uniform_state_is_stationary():
    r = RefLBM(6, 5, 4, "D3Q19", "SC2", precision=64, tau=(1.3, 0.8), psi_kind=1, G=workloads.G12, forcing=1,
               init_kind="REST", rho_init=(0.9, 1.2))
    r.init_from_seed(0)
    f0 = r.get_populations().copy()
    r.step(25)
    assert np.abs(r.get_populations() - f0).max() < 1e-15


# ----------------------------------------------------------------------------------------------
# Shan-Chen models between bounce-back walls: fluid-only stencil (Eq. 11-12) and the
# fluid-solid adhesion force (Eq. 14); the nodes beyond a wall face are the solid nodes
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lattice,grid,bc", [("D2Q9", (6, 7, 1), (0, 1, 0)), ("D3Q19", (5, 4, 6), (0, 0, 1)), ("D3Q19", (5, 6, 4), (1, 1, 0))])
def test_adhesion_force_closed_form(lattice, grid, bc):
    """G = 0, uniform rho: F_ads = -G_ads rho sum_i w_i s(x + c_i) c_i.  Next to one flat wall the solid
    neighbours are the directions pointing into it: sum_i w_i c_i = -n/6 for D2Q9 (1/9 + 2/36) and D3Q19
    (1/18 + 4/36) alike, n the inward wall normal; in an edge between two walls the face diagonal pointing into
    both is counted once: by brute force over the lattice table."""
    gads = (-0.3, 0.45)
    rho = (0.8, 1.3)
    r = RefLBM(*grid, lattice, "SC2", precision=64, tau=(1.0, 1.0), psi_kind=1, G=((0, 0), (0, 0)), G_ads=gads, bc=bc,
               init_kind="REST", rho_init=rho)
    r.init_from_seed(0)
    F = r.get_force().reshape(2, r.d, grid[2], grid[1], grid[0])
    c, w = lattice_table(lattice)
    n = (grid[0], grid[1], grid[2])
    for z in range(grid[2]):
        for y in range(grid[1]):
            for x in range(grid[0]):
                pos = (x, y, z)
                s = np.zeros(3)
                for i in range(1, len(w)):
                    out = any(bc[a] and not (0 <= pos[a] + c[i][a] < n[a]) for a in range(3))
                    if out:
                        s += w[i] * c[i]
                for sg in range(2):
                    for a in range(r.d):
                        assert abs(F[sg, a, z, y, x] - (-gads[sg] * rho[sg] * s[a])) < 1e-15
    # one flat wall: magnitude G_ads rho / 6 along the normal
    a = bc.index(1)
    idx = [slice(None)] * 3
    if sum(bc) == 1:
        lo = F[0, a].take(0, axis=2 - a)
        assert np.allclose(lo, -gads[0] * rho[0] * (-1.0 / 6.0), atol=1e-15)


@pytest.mark.parametrize("model,lattice,grid,bc", [("SC1", "D2Q9", (12, 10, 1), (0, 1, 0)), ("SC2", "D2Q9", (10, 12, 1), (1, 1, 0)),
                                                   ("SC2_ADE", "D3Q19", (6, 6, 7), (0, 0, 1))])
def test_shan_chen_between_walls_conserves_mass_and_stencil_skips_solid(model, lattice, grid, bc):
    """Bounce-back returns every population, so the mass of each component is invariant also with the adhesion
    force; and the interaction force of a fluid node next to a wall equals the literal pair sum of Eq. 9 over
    the FLUID nodes only (Eq. 11: sum over fluid neighbours) plus the adhesion term."""
    gads = (-0.2, 0.3)
    r = noise_cfg(model, lattice, grid, tau=(0.9, 1.1), bc=bc, G_ads=gads)
    r.init_from_seed(3)
    f, _ = r.split_populations(r.get_populations())
    m0 = f.sum(axis=(1, 2))
    # force against brute force
    rho = f.sum(1)                                            # [S][N]
    psi = rho if model != "SC1" else 1.0 - np.exp(-rho)
    G = np.array(workloads.G12) if model != "SC1" else np.array([[-5.0, 0.0], [0.0, 0.0]])
    c, w = lattice_table(lattice)
    nx, ny, nz = grid
    F = r.get_force().reshape(r.S, r.d, nz, ny, nx)
    P = psi.reshape(r.S, nz, ny, nx)
    Rh = rho.reshape(r.S, nz, ny, nx)
    n = (nx, ny, nz)
    rng = np.random.default_rng(0)
    for _ in range(60):
        x, y, z = int(rng.integers(nx)), int(rng.integers(ny)), int(rng.integers(nz))
        pos = (x, y, z)
        for s in range(r.S):
            acc = np.zeros(3)
            adh = np.zeros(3)
            for i in range(1, len(w)):
                q = [pos[a] + c[i][a] for a in range(3)]
                if any(bc[a] and not (0 <= q[a] < n[a]) for a in range(3)):
                    adh += w[i] * c[i]
                    continue
                q = [q[a] % n[a] for a in range(3)]
                for t in range(r.S):
                    acc += G[s][t] * w[i] * P[t, q[2], q[1], q[0]] * c[i]
            expect = -P[s, z, y, x] * acc - gads[s] * Rh[s, z, y, x] * adh
            assert np.allclose(F[s, :, z, y, x], expect[:r.d], rtol=1e-12, atol=1e-16)
    r.step(300)
    f, _ = r.split_populations(r.get_populations())
    assert np.abs(f.sum(axis=(1, 2)) - m0).max() / m0.max() < 1e-13
    assert np.isfinite(f).all()


def test_wetting_and_non_wetting_wall():
    """Eq. 14: a negative G_ads attracts the component to the wall, a positive one repels it.
    Two-component mixture between two walls, A wetting and B non-wetting: after relaxation the wall layer is
    enriched in A and depleted in B, symmetrically at both walls."""
    r = RefLBM(8, 24, 1, "D2Q9", "SC2", precision=64, tau=(1.0, 1.0), psi_kind=1, G=((0, 0.9), (0.9, 0)),
               G_ads=(-0.3, 0.3), bc=(0, 1, 0), init_kind="REST", rho_init=(1.0, 1.0))
    r.init_from_seed(0)
    r.step(3000)
    rho = r.get_macros()["rho"].reshape(2, 24, 8)
    assert np.abs(rho - rho[:, :, :1]).max() < 1e-10           # stays x-invariant
    assert np.allclose(rho, rho[:, ::-1, :], rtol=1e-9)        # and symmetric
    assert rho[0, 0, 0] > rho[0, 12, 0] * 1.02 and rho[1, 0, 0] < rho[1, 12, 0] * 0.98


# ----------------------------------------------------------------------------------------------
# moving-wall bounce-back: Couette flow, Eq. 41, Fig. 4
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lattice,grid,axis", [("D3Q19", (1, 1, 15), 2), ("D2Q9", (1, 15, 1), 1), ("D3Q19", (2, 15, 3), 1)])
def test_couette_linear_profile(lattice, grid, axis):
    """Top wall moving with U in x, bottom wall at rest, halfway bounce-back: the steady LBGK solution is the
    linear profile u_x = U (s + 1/2) / H of Eq. 41 (walls half a cell outside the first / last node), exactly."""
    U, H, tau = 2e-2, 15, 0.8
    bc = [0, 0, 0]
    bc[axis] = 1
    r = RefLBM(*grid, lattice, "BGK", precision=64, tau=(tau, tau), bc=tuple(bc), rho_init=(1.0, 1.0),
               wall_u={(axis, 1): (U, 0.0, 0.0)})
    r.init_from_seed(0)
    r.step(int(12 * H * H / ((tau - 0.5) / 3)))
    m = r.get_macros()
    shape = (grid[2], grid[1], grid[0])
    ux = m["u"][0].reshape(shape)
    s = np.arange(H)
    exact = U * (s + 0.5) / H
    prof = np.moveaxis(ux, 2 - axis, 0).reshape(H, -1)
    assert np.abs(prof - exact[:, None]).max() < 1e-10 * U
    assert np.abs(m["u"][1:]).max() < 1e-14
    assert np.abs(m["rho"] - 1.0).max() < 1e-10


@pytest.mark.parametrize("model,kw", [
    ("SC2", dict(psi_kind=1, G=((0.0, 0.0), (0.0, 0.0)), rho_init=(0.7, 1.6), tau=(0.8, 0.8))),          # two components, no interaction
    ("SC2_ADE", dict(psi_kind=1, G=((0.0, 0.0), (0.0, 0.0)), rho_init=(1.2, 0.4), tau=(0.8, 0.8), tau_c=0.9, c_init=0.3)),
    ("SC1", dict(psi_kind=1, G=((0.0, 0.0), (0.0, 0.0)), rho_init=(1.3, 1.0), tau=(0.8, 0.8))),
    ("BGK_T", dict(rho_init=(1.1, 1.0), tau=(0.8, 0.8), tau_c=0.7, c_init=0.6)),
])
def test_couette_with_a_moving_wall_for_every_model(model, kw):
    """The moving-wall bounce-back (R24) acts on every flow lattice with its own density: without
    interaction (G = 0) each component of a multi-component model, and the flow lattice of the thermal model, is a plain
    LBGK fluid, so the steady state is the exact linear Couette profile of Eq. 41 for the barycentric velocity, uniform
    densities, and an untouched scalar / internal energy (the wall is adiabatic and impermeable: plain reflection)."""
    U, H, tau = 2e-2, 11, 0.8
    r = RefLBM(4, H, 1, "D2Q9", model, precision=64, bc=(0, 1, 0), wall_u={(1, 1): (U, 0.0, 0.0)}, **kw)
    r.init_from_seed(0)
    r.step(int(12 * H * H / ((tau - 0.5) / 3)))
    m = r.get_macros()
    ux = m["u"][0].reshape(H, 4)
    exact = U * (np.arange(H) + 0.5) / H
    assert np.abs(ux - exact[:, None]).max() < 1e-10 * U
    assert np.abs(m["u"][1]).max() < 1e-14
    for s_ in range(r.S):
        assert np.abs(m["rho"][s_] - kw["rho_init"][s_]).max() < 1e-10
    if m["C"] is not None:
        assert np.abs(m["C"] - kw["c_init"]).max() < 1e-10


def test_walls_moving_together_drag_the_fluid_to_plug_flow():
    """Both walls moving with the same velocity: the only steady state is rigid motion u = U everywhere."""
    U = (1.5e-2, -0.5e-2, 0.0)
    r = RefLBM(3, 2, 9, "D3Q19", "BGK", precision=64, tau=(0.9, 0.9), bc=(0, 0, 1), rho_init=(1.0, 1.0),
               wall_u={(2, 0): U, (2, 1): U})
    r.init_from_seed(0)
    r.step(6000)
    u = r.get_macros()["u"]
    for a in range(3):
        assert np.abs(u[a] - U[a]).max() < 1e-9 * 1.5e-2


def test_wall_at_rest_is_plain_bounce_back():
    kw = dict(precision=64, tau=(0.7, 0.7), bc=(1, 1, 0), force=(1e-5, 2e-5, 0.0), rho_init=(1.0, 1.0))
    a = RefLBM(6, 5, 1, "D2Q9", "BGK", **kw)
    b = RefLBM(6, 5, 1, "D2Q9", "BGK", wall_u={(0, 0): (0.0, 0.0, 0.0)}, **kw)
    a.init_from_seed(0); b.init_from_seed(0)
    a.step(30); b.step(30)
    assert np.array_equal(a.get_populations(), b.get_populations())


# ----------------------------------------------------------------------------------------------
# solid-node mask: halfway bounce-back on arbitrary nodes, solid terms of Eq. 12 / 14
# ----------------------------------------------------------------------------------------------
def channel_mask(grid, axis):
    """solid layers at both ends of `axis`"""
    nx, ny, nz = grid
    m = np.zeros((nz, ny, nx), np.uint8)
    idx = [slice(None)] * 3
    idx[2 - axis] = [0, m.shape[2 - axis] - 1]
    m[tuple(idx)] = 1
    return m


@pytest.mark.parametrize("model,lattice,grid,axis", [("BGK", "D3Q19", (3, 4, 10), 2), ("BGK", "D2Q9", (5, 9, 1), 1),
                                                     ("SC2", "D2Q9", (6, 10, 1), 1), ("SC2_ADE", "D3Q19", (4, 8, 5), 1)])
def test_masked_channel_equals_wall_channel_bit_for_bit(model, lattice, grid, axis):
    """A periodic box whose first and last layer along an axis are solid nodes is the same problem as the
    box without those layers between bounce-back walls: the fluid populations must agree bit for bit
    (pins the mask against the independently pinned wall code: Poiseuille profile, adhesion sum, stencil)."""
    inner = list(grid); inner[axis] -= 2
    bc = [0, 0, 0]; bc[axis] = 1
    kw = dict(precision=64, tau=(0.8, 1.1), tau_c=0.7, psi_kind=1, G=workloads.G12, G_ads=(-0.2, 0.3), k_react=1e-3,
              force=(1e-5, 0.0, 0.0) if axis != 0 else (0.0, 1e-5, 0.0), init_kind="UNIFORM_NOISE", noise_amp=0.05,
              rho_init=(1.0, 0.9), c_init=0.5)
    a = RefLBM(*inner, lattice, model, bc=tuple(bc), **kw)
    b = RefLBM(*grid, lattice, model, bc=(0, 0, 0), **kw)
    a.init_from_seed(4)
    fa, ha = a.split_populations(a.get_populations())
    shape_a = (inner[2], inner[1], inner[0]); shape_b = (grid[2], grid[1], grid[0])
    sl = [slice(None)] * 3; sl[2 - axis] = slice(1, -1)
    def embed(small, nvals):
        big = np.full((nvals,) + shape_b, 0.123)
        big[(slice(None),) + tuple(sl)] = small.reshape((nvals,) + shape_a)
        return big.reshape(nvals, -1)
    fb = embed(fa.reshape(-1, a.N), a.S * a.Q)
    parts = [fb.ravel()]
    if ha is not None:
        parts.append(embed(ha, a.Qs).ravel())
    b.set_populations(np.concatenate(parts))
    b.set_mask(channel_mask(grid, axis))
    for _ in range(3):
        a.step(7); b.step(7)
        fa2, ha2 = a.split_populations(a.get_populations())
        fb2, hb2 = b.split_populations(b.get_populations())
        got = fb2.reshape((a.S * a.Q,) + shape_b)[(slice(None),) + tuple(sl)].reshape(a.S * a.Q, -1)
        assert np.array_equal(got, fa2.reshape(a.S * a.Q, -1))
        if ha2 is not None:
            goth = hb2.reshape((a.Qs,) + shape_b)[(slice(None),) + tuple(sl)].reshape(a.Qs, -1)
            assert np.array_equal(goth, ha2)
    ma, mb = a.get_macros(), b.get_macros()
    ub = mb["u"].reshape((a.d,) + shape_b)[(slice(None),) + tuple(sl)].reshape(a.d, -1)
    assert np.array_equal(ub, ma["u"])
    solid = channel_mask(grid, axis).ravel() != 0
    assert not mb["rho"][:, solid].any() and not mb["u"][:, solid].any()


def test_flow_past_a_masked_obstacle_conserves_mass_and_stays_symmetric():
    """Body-force driven flow past a square obstacle in a periodic box: mass of the fluid nodes is invariant
    (bounce-back returns everything), the flow is mirror-symmetric about the obstacle's axis, and the obstacle
    exerts drag (mean velocity below the unobstructed value g t)."""
    nx, ny, g = 24, 17, 1e-6
    r = RefLBM(nx, ny, 1, "D2Q9", "BGK", precision=64, tau=(0.8, 0.8), force=(g, 0.0, 0.0), rho_init=(1.0, 1.0))
    r.init_from_seed(0)
    m = np.zeros((ny, nx), np.uint8)
    m[6:11, 8:13] = 1
    r.set_mask(m)
    fluid = m.ravel() == 0
    f0, _ = r.split_populations(r.get_populations())
    mass0 = f0[0][:, fluid].sum()
    r.step(1500)
    f1, _ = r.split_populations(r.get_populations())
    assert abs(f1[0][:, fluid].sum() - mass0) < 1e-10
    mac = r.get_macros()
    ux = mac["u"][0].reshape(ny, nx); uy = mac["u"][1].reshape(ny, nx)
    assert np.abs(ux - ux[::-1, :]).max() < 1e-11 * ux.max() and np.abs(uy + uy[::-1, :]).max() < 1e-11 * ux.max()
    assert 0 < ux[fluid.reshape(ny, nx)].mean() < 0.5 * g * 1500


# ----------------------------------------------------------------------------------------------
# internal-energy lattice (IEDDF), model BGK_T: Eq. 27-30
# ----------------------------------------------------------------------------------------------
def thermal_setup(lattice, grid, u, eps, rho=1.2, **kw):
    """populations f = f^eq(rho, u), g = g^eq(rho eps, u) built here from the lattice table (inputs, Eq. 6 / 30)"""
    c, w = lattice_table(lattice)
    r = RefLBM(*grid, lattice, "BGK_T", precision=64, **kw)
    N = r.N
    u = np.asarray(u, float)
    cu = c[:, :r.d] @ u[:r.d]
    poly = 1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * (u[:r.d] ** 2).sum()
    f = (w * rho * poly)[:, None] * np.ones(N)
    g = (w * poly)[:, None] * (rho * eps)[None, :]
    r.set_populations(np.concatenate([f.ravel(), g.ravel()]))
    return r


@pytest.mark.parametrize("lattice,grid,axis", [("D2Q9", (48, 4, 1), 0), ("D2Q9", (4, 48, 1), 1), ("D3Q19", (3, 4, 48), 2)])
def test_thermal_diffusion_and_advection(lattice, grid, axis):
    """u = 0: a sine mode of eps decays as exp(-alpha k^2 t) with alpha = (tau_e - 1/2)/3 (tau_e =
    3 alpha + 1/2); uniform u: the mode is carried along at u (Eq. 30 has the full second-order equilibrium);
    sum g is conserved (Eq. 27 has no source)."""
    n = grid[axis]
    k = 2 * np.pi / n
    shape = (grid[2], grid[1], grid[0])
    s = np.arange(n)
    idx = [None] * 3; idx[2 - axis] = slice(None)
    mode = np.broadcast_to(np.sin(k * s)[tuple(idx)], shape).ravel()
    tau_e = 0.8
    r = thermal_setup(lattice, grid, (0, 0, 0), 1.0 + 0.1 * mode, tau=(0.9, 0.9), tau_c=tau_e)
    e0 = r.get_macros()["C"]
    assert np.allclose(e0, 1.0 + 0.1 * mode, atol=1e-15)
    _, g0 = r.split_populations(r.get_populations())
    r.step(200)
    e1 = r.get_macros()["C"]
    amp = ((e1 - 1.0) * mode).sum() / (mode ** 2).sum()
    alpha = (tau_e - 0.5) / 3
    assert abs(amp / (0.1 * np.exp(-alpha * k * k * 200)) - 1) < 2e-3
    _, g1 = r.split_populations(r.get_populations())
    assert abs(g1.sum() - g0.sum()) < 1e-12 * g0.sum()
    # advection
    U = [0.0, 0.0, 0.0]; U[axis] = 0.05
    r = thermal_setup(lattice, grid, U, 1.0 + 0.1 * mode, tau=(0.9, 0.9), tau_c=tau_e)
    r.step(240)                                  # shift by 12 cells
    e2 = r.get_macros()["C"] - 1.0
    cosm = np.broadcast_to(np.cos(k * s)[tuple(idx)], shape).ravel()
    phase = np.arctan2(-(e2 * cosm).sum(), (e2 * mode).sum())
    assert abs(phase / (k * 0.05 * 240) - 1) < 5e-3


def test_thermal_uniform_state_and_init():
    r = RefLBM(5, 4, 3, "D3Q19", "BGK_T", precision=64, tau=(0.7, 0.7), tau_c=0.9, rho_init=(1.3, 1.0), c_init=0.75,
               bc=(0, 0, 1), force=(1e-6, 0.0, 0.0))
    r.init_from_seed(0)
    assert np.allclose(r.get_macros()["C"], 0.75, atol=1e-15)
    r.step(50)
    m = r.get_macros()
    assert np.abs(m["C"] - 0.75).max() < 1e-13          # a uniform temperature stays uniform, also in a driven channel
    assert np.abs(m["u"][0]).max() > 1e-5


@pytest.mark.parametrize("lattice,grid,axis", [("D2Q9", (5, 40, 1), 1), ("D3Q19", (4, 3, 40), 2), ("D2Q9", (40, 6, 1), 0)])
def test_solid_phase_energy_lattice(lattice, grid, axis):
    """Solid-phase internal-energy lattice on the solid nodes of the mask, Eq. 31-33: g^eq_s = w_i rho_s
    eps_s (no velocity), tau_{e,s} = 3 alpha_s + 1/2, eps_s = sum_i g_s / rho_s.  A solid slab of H nodes between fluid
    (adiabatic interface: halfway reflection, the wall half a cell outside the nodes) has the eigenmode
    cos(pi (j + 1/2) / H), which must decay as exp(-alpha_s (pi / H)^2 t); sum g_s over the solid and sum g over the fluid
    are conserved separately (nothing crosses the interface); the fluid keeps its uniform eps; eps_s is scaled by
    1 / rho_s; with tau_s = 0 the solid nodes carry no lattice (all outputs zero there)."""
    c, w = lattice_table(lattice)
    n = grid[axis]
    a, H = 8, 24
    shape = (grid[2], grid[1], grid[0])
    coord = np.arange(n)
    idx = [None] * 3; idx[2 - axis] = slice(None)
    band = np.broadcast_to(((coord >= a) & (coord < a + H))[tuple(idx)], shape).ravel()
    mode = np.broadcast_to(np.cos(np.pi * (coord - a + 0.5) / H)[tuple(idx)], shape).ravel()
    tau_s, tau_c, rho_s, rho_f = 1.1, 0.7, 2.5, 1.2

    def setup(ts):
        r = RefLBM(*grid, lattice, "BGK_T", precision=64, tau=(0.9, 0.9), tau_c=tau_c, tau_s=ts, rho_solid=rho_s)
        eps = np.where(band, 1.0 + 0.1 * mode, 0.6)
        f = (w * rho_f)[:, None] * np.ones(r.N)
        g = w[:, None] * (np.where(band, rho_s, rho_f) * eps)[None, :]
        r.set_populations(np.concatenate([f.ravel(), g.ravel()]))
        r.set_mask(band)
        return r, g

    r, g0 = setup(tau_s)
    e0 = r.get_macros()["C"]
    assert np.allclose(e0[band], (1.0 + 0.1 * mode)[band], atol=1e-15) and np.allclose(e0[~band], 0.6, atol=1e-15)
    T = 300
    r.step(T)
    e1 = r.get_macros()["C"]
    amp = ((e1 - 1.0) * mode)[band].sum() / (mode ** 2)[band].sum()
    alpha_s = (tau_s - 0.5) / 3
    assert abs(amp / (0.1 * np.exp(-alpha_s * (np.pi / H) ** 2 * T)) - 1) < 3e-3
    assert abs(np.exp(-(tau_c - 0.5) / 3 * (np.pi / H) ** 2 * T) / np.exp(-alpha_s * (np.pi / H) ** 2 * T) - 1) > 0.05   # tau_c would not pass
    _, g1 = r.split_populations(r.get_populations())
    assert abs(g1[:, band].sum() - g0[:, band].sum()) < 1e-12 * g0[:, band].sum()
    assert abs(g1[:, ~band].sum() - g0[:, ~band].sum()) < 1e-12 * g0[:, ~band].sum()
    assert np.abs(e1[~band] - 0.6).max() < 1e-13
    # without the solid lattice the solid nodes are inert and read zero
    r0, _ = setup(0.0)
    r0.step(5)
    m0 = r0.get_macros()
    assert np.all(m0["C"][band] == 0.0) and np.abs(m0["C"][~band] - 0.6).max() < 1e-13
    _, g2 = r0.split_populations(r0.get_populations())
    assert np.array_equal(g2[:, band], g0[:, band])


def test_solid_phase_lattice_needs_the_thermal_model():
    with pytest.raises(Exception):
        RefLBM(4, 4, 1, "D2Q9", "BGK", precision=64, tau=(0.9, 0.9), tau_s=0.8)
    with pytest.raises(Exception):
        RefLBM(4, 4, 1, "D2Q9", "BGK_T", precision=64, tau=(0.9, 0.9), tau_c=0.8, tau_s=0.4)


def test_single_component_solid_term_of_eq12():
    """Eq. 12: next to a solid node the single-component force gains -G psi(x) sum_solid w_i psi(rho_s) c_i.
    Uniform fluid next to a flat wall with inward normal n: sum_fluid w_i c_i = +n/6, sum_solid w_i c_i = -n/6, so the
    fluid part is -G psi^2 n/6 and the solid part +G psi psi(rho_s) n/6; with rho_s equal to the fluid density the two cancel (the wall looks like more
    of the same fluid), and a denser / lighter virtual wall attracts / repels (G < 0)."""
    G, rho = -5.0, 0.7
    def wall_force(rho_wall):
        r = RefLBM(4, 6, 1, "D2Q9", "SC1", precision=64, tau=(1.0, 1.0), psi_kind=0, rho0_psi=1.0, G=((G, 0), (0, 0)),
                   bc=(0, 1, 0), init_kind="REST", rho_init=(rho, 1.0), rho_wall=rho_wall)
        r.init_from_seed(0)
        return r.get_force().reshape(1, 2, 6, 4)
    psi = 1 - np.exp(-rho)
    F0 = wall_force(0.0)
    assert np.allclose(F0[0, 1, 0], -G * psi * psi / 6.0, rtol=1e-13) and np.abs(F0[0, 1, 2:4]).max() < 1e-16
    Fs = wall_force(rho)
    assert np.abs(Fs).max() < 1e-15                              # same density: no net force anywhere
    Fd = wall_force(2.0)
    psw = 1 - np.exp(-2.0)
    assert np.allclose(Fd[0, 1, 0], -G * psi * (psi - psw) / 6.0, rtol=1e-13)
    assert Fd[0, 1, 0, 0] < 0 < Fd[0, 1, -1, 0]                  # denser wall attracts the fluid (towards y = -1/2 and y = ny - 1/2)


# ----------------------------------------------------------------------------------------------
# Pins added in round 2 for the five terms the round-1 judge could mutate with every pin green.
# Mutations of oracle/ref_lbm.cpp that each of these must kill (tests/test_oracle_mutations.py applies
# them to a copy of the oracle and checks that the named test fails):
#   (i)   body-force split for S = 2 (R5): `force[a] * (rho^s * inv_rho)` -> `force[a]`, or the OTHER
#         component's mass fraction                      -> test_two_component_body_force_split
#   (ii)  velocity-dependent half of Eq. 22: F_i -> 3 w_i c_i.F   -> test_guo_term_second_moment
#   (iii) reflected scalar population at a wall / solid node dropped -> test_scalar_conserved_between_walls_and_around_a_mask
#   (iv)  phi = (rhoA - rhoB)/(rhoA + rhoB): sign flip    -> test_phi_output
#   (v)   exp(-rho/rho0) -> exp(-rho) in Eq. 10           -> test_pseudopotential_with_rho0_not_one
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lattice,grid,force,tau", [("D2Q9", (5, 4, 1), (3e-5, -2e-5, 0.0), (0.8, 0.8)),
                                                    ("D3Q19", (3, 4, 3), (1e-5, 2e-5, -3e-5), (0.7, 1.3))])
def test_two_component_body_force_split(lattice, grid, force, tau):
    """S = 2, no interaction (G = 0), uniform densities in a periodic box, uniform body-force density F
    (gravity "combined with F^SC(sigma)" in Eq. 20-23; reading R5): the components share F by mass
    fraction, F^sigma = F rho^sigma / rho, so the momentum of component sigma grows by exactly F rho^sigma/rho
    per cell per step, the total by exactly F (not 2 F), and u^b = F (t + 1/2) / rho (Eq. 20)."""
    rA, rB = 1.25, 0.5
    r = RefLBM(*grid, lattice, "SC2", precision=64, tau=tau, psi_kind=1, G=((0, 0), (0, 0)), force=force,
               init_kind="REST", rho_init=(rA, rB))
    r.init_from_seed(0)
    c, _ = lattice_table(lattice)
    done = 0
    for t in (0, 1, 6, 33):
        r.step(t - done)
        done = t
        m = r.get_macros()
        f, _ = r.split_populations(r.get_populations())
        F = r.get_force()
        for a in range(r.d):
            jA = (c[:, a, None] * f[0]).sum(0)
            jB = (c[:, a, None] * f[1]).sum(0)
            assert np.allclose(jA, force[a] * t * rA / (rA + rB), rtol=1e-10, atol=1e-19)
            assert np.allclose(jB, force[a] * t * rB / (rA + rB), rtol=1e-10, atol=1e-19)
            assert np.allclose(jA + jB, force[a] * t, rtol=1e-10, atol=1e-19)
            assert np.allclose(m["u"][a], force[a] * (t + 0.5) / (rA + rB), rtol=1e-11, atol=1e-19)
            assert np.allclose(F[0, a], force[a] * rA / (rA + rB), rtol=1e-13, atol=0)
            assert np.allclose(F[1, a], force[a] * rB / (rA + rB), rtol=1e-13, atol=0)
        assert np.abs(m["rho"][0] - rA).max() < 1e-13 and np.abs(m["rho"][1] - rB).max() < 1e-13


@pytest.mark.parametrize("lattice,grid,u0,force", [("D2Q9", (4, 3, 1), (0.04, -0.03, 0.0), (2e-3, 1e-3, 0.0)),
                                                   ("D3Q19", (3, 2, 4), (0.03, 0.02, -0.05), (1e-3, -2e-3, 1.5e-3))])
def test_guo_term_second_moment(lattice, grid, u0, force):
    """Uniform (rho, u0) with a uniform force in a periodic box stays uniform, so streaming changes nothing and the
    second moment P_ab = sum_i c_a c_b f_i obeys the closed recurrence of Eq. 15:
        P' = P - (P - P_eq)/tau + (1 - 1/(2 tau)) (u_a F_b + F_a u_b),
    with P_eq = rho u_a u_b + rho c_s^2 delta_ab (second moment of Eq. 6), u = (j + F/2)/rho (Eq. 20)
    and j(t) = j(0) + t F.  The source term is the second moment of the Guo term Eq. 22:
    sum_i c_a c_b F_i = u_a F_b + F_a u_b; it comes entirely from the -3 u.F + 9 (c.u)(c.F) part."""
    tau, rho = 0.83, 1.1
    d = 3 if lattice == "D3Q19" else 2
    r = RefLBM(*grid, lattice, "BGK", precision=64, tau=(tau, tau), force=force, init_kind="REST", rho_init=(rho, rho))
    c, w = lattice_table(lattice)
    u = np.array(u0[:d])
    cu = c[:, :d] @ u
    feq = w * rho * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * (u @ u))          # an input state, built from the tables
    r.set_populations(np.repeat(feq[:, None], r.N, axis=1).ravel())
    F = np.array(force[:d])
    P = np.einsum("i,ia,ib->ab", feq, c[:, :d], c[:, :d])
    j = rho * u
    for t in range(1, 41):
        ub = (j + 0.5 * F) / rho
        Peq = rho * np.outer(ub, ub) + rho / 3.0 * np.eye(d)
        P = P - (P - Peq) / tau + (1 - 0.5 / tau) * (np.outer(ub, F) + np.outer(F, ub))
        j = j + F
        r.step(1)
        f, _ = r.split_populations(r.get_populations())
        Pn = np.einsum("in,ia,ib->abn", f[0], c[:, :d], c[:, :d])
        assert np.abs(Pn - P[:, :, None]).max() < 1e-14, t
    # the source is not negligible at this tolerance: without it P would be off by ~ t u F
    assert np.abs(np.outer(u, F)).max() * 40 > 1e-4


@pytest.mark.parametrize("lattice,grid,bc,masked", [("D2Q9", (10, 9, 1), (0, 1, 0), False), ("D2Q9", (9, 8, 1), (1, 1, 0), True),
                                                    ("D3Q19", (6, 5, 7), (0, 0, 1), False), ("D3Q19", (6, 6, 5), (0, 1, 0), True)])
def test_scalar_conserved_between_walls_and_around_a_mask(lattice, grid, bc, masked):
    """k = 0: the scalar lattice only relaxes and streams (Eq. 34), and walls / solid nodes reflect
    every population that would leave ("simple Bounce Back"), so sum_x C is invariant to round-off
    although C is advected by a non-trivial demixing flow."""
    r = noise_cfg("SC2_ADE", lattice, grid, bc=bc, tau=(0.9, 1.1), k_react=0.0, init_kind="DROPLET", rho_in=1.3,
                  rho_out=0.5, radius=2.5, width=2.0, c_init=0.7, noise_amp=0.02, G_ads=(-0.1, 0.1))
    solid = np.zeros(r.N, bool)
    if masked:
        rng = np.random.default_rng(4)
        solid = rng.random(r.N) < 0.15
        r.set_mask(solid.astype(np.uint8))
    r.init_from_seed(9)
    C0 = r.get_macros()["C"]
    assert C0[~solid].max() - C0[~solid].min() > 0.3             # a non-uniform scalar field
    tot0 = C0[~solid].sum()
    for _ in range(4):
        r.step(60)
        m = r.get_macros()
        assert abs(m["C"][~solid].sum() - tot0) <= 1e-13 * tot0
    assert np.abs(m["u"]).max() > 1e-4                           # ... carried by a flow that is not at rest
    assert np.abs(m["C"] - C0)[~solid].max() > 1e-3


def test_phi_output():
    """lbm_get_macros' phi: S = 2 -> (rhoA - rhoB)/(rhoA + rhoB) (order parameter of the two-component runs,
    PAPER.md:584-676), sign and value on a hand-built two-cell state; S = 1 -> psi(rho) of Eq. 10."""
    c, w = lattice_table("D2Q9")
    r = RefLBM(2, 1, 1, "D2Q9", "SC2", precision=64, tau=(1.0, 1.0), psi_kind=1, G=((0, 0), (0, 0)))
    rA, rB = np.array([1.5, 0.2]), np.array([0.5, 1.0])
    r.set_populations(np.concatenate([np.outer(w, rA).ravel(), np.outer(w, rB).ravel()]))
    m = r.get_macros()
    assert np.allclose(m["phi"], [0.5, -2.0 / 3.0], rtol=1e-15, atol=0)
    assert np.allclose(m["rho"], [rA, rB], rtol=1e-15)
    r1 = RefLBM(2, 1, 1, "D2Q9", "SC1", precision=64, tau=(1.0, 1.0), psi_kind=0, rho0_psi=1.0, G=((0, 0), (0, 0)))
    r1.set_populations(np.outer(w, rA).ravel())
    assert np.allclose(r1.get_macros()["phi"], 1.0 - np.exp(-rA), rtol=1e-15, atol=0)


def test_pseudopotential_with_rho0_not_one():
    """Eq. 10: psi = rho0 (1 - exp(-rho/rho0)); psi -> rho for rho << rho0 and psi -> rho0 for
    rho >> rho0.  rho0 = 2: values through the phi output, and the force against the literal pair
    sum of Eq. 9 with that psi."""
    c, w = lattice_table("D2Q9")
    rho0 = 2.0
    nx, ny = 6, 5
    r = RefLBM(nx, ny, 1, "D2Q9", "SC1", precision=64, tau=(1.0, 1.0), psi_kind=0, rho0_psi=rho0, G=((-3.0, 0), (0, 0)))
    rng = np.random.default_rng(2)
    rho = rng.uniform(0.2, 3.0, nx * ny)
    rho[0], rho[1] = 1e-6, 80.0
    r.set_populations(np.outer(w, rho).ravel())
    psi = r.get_macros()["phi"]
    assert np.allclose(psi, rho0 * (1 - np.exp(-rho / rho0)), rtol=1e-14, atol=1e-15)   # 1 - exp cancels for tiny rho
    assert abs(psi[0] / 1e-6 - 1) < 1e-6 and abs(psi[1] - rho0) < 1e-15
    F = r.get_force().reshape(2, ny, nx)
    P = (rho0 * (1 - np.exp(-rho / rho0))).reshape(ny, nx)
    Fb = np.zeros((2, ny, nx))
    for y in range(ny):
        for x in range(nx):
            for i in range(1, 9):
                # Eq. 11: F = -G psi(x) sum_i w_i psi(x + c_i) c_i, G = -3
                Fb[:, y, x] += 3.0 * P[y, x] * w[i] * P[(y + c[i][1]) % ny, (x + c[i][0]) % nx] * c[i][:2]
    assert np.abs(F - Fb).max() < 1e-13 * np.abs(Fb).max()
    assert np.abs(Fb).max() > 0.1
