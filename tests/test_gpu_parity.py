"""Parity of the CUDA library (through the C ABI of include/lbm.h) with the CPU oracle.  `-m gpu`.

Same seeded inputs on both sides (workloads.py); the oracle never sees a value produced by the
CUDA path.  Bars:
  * populations, models without a transcendental (BGK, psi = rho): BIT-EXACT, fp64 and fp32 --
    both sides evaluate the same IEEE expression tree without FMA contraction;
  * SC1 (psi = 1 - exp(-rho), Eq. 10): CUDA's and glibc's exp differ by <= 1 ulp, so <= 1e-13
    per field over 16 steps and the north-star bar <= 1e-12 (fp64) after 1000 steps;
  * fields after 1000 steps: max|a-b| / max|b| <= 1e-12 (fp64), <= 1e-5 (fp32 vs fp32 oracle),
    vector fields with the Euclidean norm per cell (BASELINE.json north_star; R14).
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def gpu():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need a B200")
    import __graft_entry__ as ge
    ge.build()                       # no-op when liblbm.so is up to date; the library itself never builds on demand
    import paper_2502_12955_b200 as lbm
    lbm.lib()
    return lbm


def make_pair(lbm, cfg):
    from oracle.ref_lbm import RefLBM
    ref = RefLBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev = lbm.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    return ref, dev


def field_err(a, b):
    """max_x |a - b| / max_x |b|; a, b shaped (components, N) or (N,): Euclidean norm over components."""
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    if a.ndim == 1:
        a, b = a[None], b[None]
    num = np.sqrt(((a - b) ** 2).sum(0)).max()
    den = np.sqrt((b ** 2).sum(0)).max()
    return num / den if den > 0 else num


def macro_errs(ref, dev):
    mr = ref.get_macros()
    md = dev.get_macros()
    out = {}
    for s in range(ref.S):
        out["rho%d" % s] = field_err(md["rho"][s].cpu().numpy(), mr["rho"][s])
    out["u"] = field_err(md["u"].cpu().numpy(), mr["u"])
    out["phi"] = field_err(md["phi"].cpu().numpy(), mr["phi"])
    if mr["C"] is not None:
        out["C"] = field_err(md["C"].cpu().numpy(), mr["C"])
    return out


SMALL = [
    # (config, grid, overrides)
    ("cfg1", (8, 8, 1), {}),
    ("cfg1", (7, 5, 1), {}),
    ("cfg1", (33, 17, 1), {}),
    ("cfg1", (9, 6, 1), dict(bc=(0, 1, 0), force=(2e-5, 0.0, 0.0))),
    ("cfg1", (6, 9, 1), dict(bc=(1, 1, 0), force=(1e-5, -2e-5, 0.0))),
    ("cfg2", (8, 8, 1), dict(radius=2.5)),
    ("cfg2", (33, 17, 1), dict(radius=5.0)),
    ("cfg3", (8, 8, 1), {}),
    ("cfg3", (33, 17, 1), dict(force=(1e-5, 2e-5, 0.0), tau=(0.8, 1.3))),
    ("cfg4", (8, 8, 8), {}),
    ("cfg4", (33, 17, 9), {}),
    ("cfg4", (5, 4, 7), dict(bc=(1, 0, 1))),
    ("cfg4", (4, 6, 5), dict(bc=(1, 1, 1), force=(1e-6, 2e-6, -1e-6))),
    ("cfg4", (8, 6, 5), dict(bc=(0, 0, 0), force=(0.0, 0.0, 0.0), init_kind="TAYLOR_GREEN", u0=0.03)),
    ("cfg4", (8, 8, 8), dict(precision=32)),
    ("cfg4", (33, 17, 9), dict(precision=32)),
    ("cfg5", (8, 8, 8), dict(rmin=2.0, rmax=3.0, vol_frac=0.2)),
    ("cfg5", (33, 17, 9), dict(rmin=2.0, rmax=4.0, vol_frac=0.1)),
    ("cfg5", (12, 9, 7), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, precision=64, tau=(0.9, 1.1), tau_c=0.7)),
    ("cfg3", (16, 8, 1), dict(precision=32)),
    # fp32 BGK with an even nx >= 64 and periodic x: the two-cells-per-thread kernel (k_step_v2)
    ("cfg4", (64, 5, 6), dict(precision=32)),
    ("cfg4", (258, 4, 3), dict(precision=32, bc=(0, 1, 1), force=(1e-6, 2e-6, -1e-6))),
    ("cfg4", (130, 6, 5), dict(precision=32, bc=(0, 0, 0), force=(0.0, 0.0, 0.0), init_kind="TAYLOR_GREEN", u0=0.03)),
    ("cfg1", (260, 9, 1), dict(precision=32)),
    ("cfg1", (66, 7, 1), dict(precision=32, bc=(0, 1, 0), force=(2e-5, 1e-5, 0.0))),
    # internal-energy lattice (model BGK_T, Eq. 27-30)
    ("cfgT", (9, 6, 7), {}),
    ("cfgT", (33, 5, 4), dict(precision=32, bc=(1, 0, 1))),
    ("cfgT2", (33, 17, 1), {}),
    ("cfgT2", (8, 9, 1), dict(bc=(0, 1, 0), force=(1e-5, 0.0, 0.0))),
    # moving-wall bounce-back (Couette, Eq. 41)
    ("cfg4", (5, 4, 7), dict(bc=(0, 0, 1), force=(0.0, 0.0, 0.0), wall_u={(2, 1): (0.02, -0.01, 0.0)})),
    ("cfg4", (6, 5, 4), dict(bc=(1, 1, 1), wall_u={(0, 0): (0.0, 0.01, 0.02), (1, 1): (0.01, 0.0, -0.01), (2, 0): (0.02, 0.01, 0.0)}, precision=32)),
    ("cfg1", (9, 6, 1), dict(bc=(0, 1, 0), wall_u={(1, 0): (-0.01, 0.0, 0.0), (1, 1): (0.03, 0.0, 0.0)})),
    # ... for the other models too (every flow lattice with its own density; scalar / energy lattices plainly reflected)
    ("cfgT", (9, 6, 7), dict(wall_u={(2, 0): (0.0, 0.02, 0.0), (2, 1): (0.03, 0.0, 0.0)})),
    ("cfgT2", (8, 9, 1), dict(bc=(1, 1, 0), force=(0.0, 0.0, 0.0), wall_u={(1, 1): (0.02, 0.0, 0.0), (0, 0): (0.0, -0.01, 0.0)}, precision=32)),
    ("cfg2", (17, 12, 1), dict(radius=4.0, bc=(0, 1, 0), G_ads=(-0.3, 0.0), wall_u={(1, 1): (0.02, 0.0, 0.0)})),
    ("cfg3", (16, 9, 1), dict(bc=(1, 1, 0), G_ads=(-0.2, 0.3), wall_u={(1, 0): (0.01, 0.0, 0.0), (0, 1): (0.0, 0.02, 0.0)})),
    ("cfg5", (12, 9, 7), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, bc=(0, 0, 1), G_ads=(-0.3, 0.3), wall_u={(2, 1): (0.02, -0.01, 0.0)})),
    # Shan-Chen models between bounce-back walls: fluid-only stencil + adhesion force (Eq. 11-12, 14)
    ("cfg2", (33, 17, 1), dict(radius=5.0, bc=(0, 1, 0), G_ads=(-0.4, 0.0))),
    ("cfg2", (17, 12, 1), dict(radius=4.0, bc=(1, 1, 0), rho_wall=1.2)),
    ("cfg3", (16, 9, 1), dict(bc=(1, 1, 0), G_ads=(-0.2, 0.3), force=(1e-5, -2e-5, 0.0))),
    ("cfg3", (9, 12, 1), dict(bc=(0, 1, 0), G_ads=(0.25, -0.25), forcing=1, tau=(0.8, 1.2))),
    ("cfg5", (12, 9, 7), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, bc=(0, 0, 1), G_ads=(-0.3, 0.3))),
    ("cfg5", (7, 6, 5), dict(rmin=1.0, rmax=2.0, vol_frac=0.2, bc=(1, 1, 1), G_ads=(0.1, -0.2), precision=64, tau=(0.9, 1.1))),
    # Shan-Chen velocity-shift forcing scheme (forcing = 1, Eq. 16-19)
    ("cfg1", (9, 6, 1), dict(forcing=1, bc=(0, 1, 0), force=(2e-5, 0.0, 0.0))),
    ("cfg1", (8, 8, 1), dict(forcing=1)),
    ("cfg2", (33, 17, 1), dict(forcing=1, radius=5.0)),
    ("cfg3", (33, 17, 1), dict(forcing=1, force=(1e-5, 2e-5, 0.0), tau=(0.8, 1.3))),
    ("cfg4", (5, 4, 7), dict(forcing=1, bc=(1, 0, 1))),
    ("cfg4", (33, 17, 9), dict(forcing=1, precision=32)),
    ("cfg5", (33, 17, 9), dict(forcing=1, rmin=2.0, rmax=4.0, vol_frac=0.1, tau=(0.9, 1.2))),
    ("cfg5", (12, 9, 7), dict(forcing=1, rmin=2.0, rmax=3.0, vol_frac=0.2, precision=64, tau=(0.9, 1.1), tau_c=0.7)),
]


@pytest.mark.parametrize("name,grid,over", SMALL, ids=lambda v: str(v).replace(" ", ""))
def test_populations_exact_steps_1_to_16(gpu, name, grid, over):
    """Population-exact comparison at every step 1..16 (odd and even AA parity), small and awkward
    grids that are not multiples of the block size, every model, walls on/off."""
    cfg = workloads.config(name, grid=grid, **over)
    ref, dev = make_pair(gpu, cfg)
    ref.init_from_seed(7)
    f0 = ref.get_populations()
    dev.set_populations(torch.from_numpy(f0))     # identical inputs: the oracle's seeded state
    exact = not (cfg["model"] == "SC1" and cfg["params"].get("psi_kind", 0) == 0)
    for step in range(1, 17):
        ref.step(1)
        dev.step(1)
        fr = ref.get_populations()
        fd = dev.get_populations().cpu().numpy()
        if exact:
            bad = np.flatnonzero(fr != fd)
            assert bad.size == 0, "step %d: %d of %d populations differ, first at %d: %r vs %r" % (
                step, bad.size, fr.size, bad[0], fd[bad[0]], fr[bad[0]])
        else:
            err = np.abs(fr - fd).max() / np.abs(fr).max()
            assert err <= 1e-13, "step %d: population error %.3e" % (step, err)
    errs = macro_errs(ref, dev)
    if ref.S == 1 and cfg["params"].get("psi_kind", 0) == 0:
        ulp = 1.2e-7 if cfg["params"]["precision"] == 32 else 2.3e-16
        assert errs.pop("phi") <= (4 * ulp if exact else 1e-13)    # phi = psi(rho) goes through exp (<= 1-2 ulp)
    tol = 0.0 if exact else 1e-13
    assert max(errs.values()) <= tol, errs
    Fr = ref.get_force()
    Fd = dev.get_force().cpu().numpy()
    if exact:
        assert np.array_equal(Fr, Fd)
    else:
        assert np.abs(Fr - Fd).max() <= 1e-13 * max(np.abs(Fr).max(), 1e-300)


@pytest.mark.parametrize("name,grid,over", [
    ("cfg1", (64, 64, 1), {}),
    ("cfg2", (40, 24, 1), dict(radius=8.0)),
    ("cfg3", (24, 40, 1), {}),
    ("cfg4", (6, 5, 16), {}),
    ("cfg4", (12, 10, 8), dict(bc=(0, 0, 0), force=(0.0, 0.0, 0.0), init_kind="TAYLOR_GREEN", u0=0.05)),
    ("cfg5", (24, 20, 16), dict(rmin=3.0, rmax=6.0, vol_frac=0.1)),
    ("cfg5", (24, 20, 1), dict(rmin=3.0, rmax=6.0, vol_frac=0.1)),
], ids=lambda v: str(v).replace(" ", ""))
def test_init_from_seed_matches_oracle(gpu, name, grid, over):
    """lbm_init_from_seed against ref_init_from_seed: the counter-based noise is integer-exact; the
    macroscopic fields go through cos/sin/tanh/sqrt in double (<= few ulp between libm and CUDA)."""
    if name == "cfg5" and grid[2] == 1:
        cfg = workloads.config(name, grid=grid, **over)
        cfg["lattice"] = "D2Q9"
    else:
        cfg = workloads.config(name, grid=grid, **over)
    ref, dev = make_pair(gpu, cfg)
    ref.init_from_seed(1234)
    dev.init_from_seed(1234)
    fr = ref.get_populations()
    fd = dev.get_populations().cpu().numpy()
    tol = 1e-14 if cfg["params"]["precision"] == 64 else 3e-7
    assert np.abs(fr - fd).max() <= tol * np.abs(fr).max()
    if cfg["params"]["init_kind"] in ("REST", "UNIFORM_NOISE"):
        assert np.array_equal(fr, fd)      # no transcendental on the way: bit-exact


def run_1000(gpu, cfg, seed, nsteps=1000):
    ref, dev = make_pair(gpu, cfg)
    ref.init_from_seed(seed)
    dev.set_populations(torch.from_numpy(ref.get_populations()))
    ref.step(nsteps)
    dev.step(nsteps)
    return ref, dev


def test_cfg1_taylor_green_1000_steps(gpu):
    """configs[0]: D2Q9 BGK fp64 64x64, 1000 steps, fields <= 1e-12 and the closed-form decay
    exp(-2 nu k^2 t), nu = (tau - 1/2)/3 (Eq. 3-6; 533-545)."""
    cfg = workloads.config("cfg1")
    ref, dev = run_1000(gpu, cfg, 1)
    errs = macro_errs(ref, dev)
    assert max(errs.values()) <= 1e-12, errs
    # the GPU path's own init + closed form, independent of the oracle
    dev.init_from_seed(1)
    dev.step(1000)
    u = dev.get_macros()["u"].cpu().numpy().reshape(2, 64, 64)
    k = 2 * np.pi / 64
    x = np.arange(64)
    mode = -np.cos(k * x)[None, :] * np.sin(k * x)[:, None]
    amp = (u[0] * mode).sum() / (mode ** 2).sum()
    exact = 0.01 * np.exp(-2 * 0.1 * k * k * 1000)
    assert abs(amp / exact - 1) <= 5e-3


def test_cfg2_shan_chen_droplet_1000_steps(gpu):
    """configs[1] at full size 256x256, R = 30, 1000 steps: fields <= 1e-12; mass conserved."""
    cfg = workloads.config("cfg2")
    ref, dev = run_1000(gpu, cfg, 2)
    errs = macro_errs(ref, dev)
    assert max(errs.values()) <= 1e-12, errs
    m0 = ref.get_macros()["rho"].sum()
    dev.step(1000)
    m1 = dev.get_macros()["rho"].double().sum().item()
    assert abs(m1 / m0 - 1) <= 1e-10


def test_cfg3_two_component_1000_steps(gpu):
    """configs[2] on a reduced 192x160 grid (the oracle needs ~3 min for 512x512), 1000 steps of
    spinodal decomposition: fields <= 1e-12 (bit-exact by construction); per-component mass."""
    cfg = workloads.config("cfg3", grid=(192, 160, 1))
    ref, dev = run_1000(gpu, cfg, 3)
    errs = macro_errs(ref, dev)
    assert max(errs.values()) <= 1e-12, errs
    rho = dev.get_macros()["rho"].cpu().numpy()
    assert np.ptp(rho[0]) > 0.05           # demixing has started (psi = rho, G12 = 1.2 > 1: R3)
    N = rho.shape[1]
    for s in range(2):
        assert abs(rho[s].sum() / N - 1.0) <= 1e-3    # +-1 % noise averages out
    m0 = rho.sum(1)
    dev.step(1000)
    m1 = dev.get_macros()["rho"].cpu().numpy().sum(1)
    assert np.abs(m1 / m0 - 1).max() <= 1e-10


@pytest.mark.parametrize("precision,tol", [(64, 1e-12), (32, 1e-5)])
def test_cfg4_poiseuille_full_size_vs_column_oracle(gpu, precision, tol):
    """configs[3] at the full 256^3 in the launch configuration bench.py times, 1000 steps, against
    the oracle run on a 1x1x256 column: the flow is x/y-invariant, which the oracle reproduces
    bit for bit (tests/test_oracle_pins.py::test_poiseuille_xy_invariance_is_bit_exact)."""
    from oracle.ref_lbm import RefLBM
    cfg = workloads.config("cfg4", precision=precision)
    col = workloads.config("cfg4", grid=(1, 1, 256), precision=precision)
    ref = RefLBM(*col["grid"], col["lattice"], col["model"], **col["params"])
    ref.init_from_seed(0)
    ref.step(1000)
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.init_from_seed(0)
    dev.step(1000)
    mr = ref.get_macros()
    md = dev.get_macros(phi=False)
    rho = md["rho"].reshape(256, 256 * 256)
    u = md["u"].reshape(3, 256, 256 * 256)
    rr = torch.from_numpy(mr["rho"].reshape(256, 1)).to(rho.device)
    ur = torch.from_numpy(mr["u"].reshape(3, 256, 1)).to(rho.device)
    e_rho = ((rho - rr).abs().max() / rr.abs().max()).item()
    e_u = (((u - ur) ** 2).sum(0).sqrt().max() / (ur ** 2).sum(0).sqrt().max()).item()
    assert e_rho <= tol and e_u <= tol, (e_rho, e_u)
    assert e_rho == 0.0 and e_u == 0.0      # same expression tree, no transcendental: bit-exact


def test_cfg4_steady_poiseuille_closed_form(gpu):
    """Guo force + halfway bounce-back on the GPU path alone against the closed form
    u_x(z) = g/(2 nu) (z+1/2)(H-z-1/2) + g/(8 nu) (16 (tau-1/2)^2/3 - 1), H = nz (DESIGN.md pins;
    PAPER.md:504-531 Eq. 43-44 with the textbook 1/2)."""
    nz, tau, g = 32, 0.9, 1e-6
    cfg = workloads.config("cfg4", grid=(16, 12, nz))
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.init_from_seed(0)
    nu = (tau - 0.5) / 3
    dev.step(int(30 * nz * nz / nu / 9.87))
    u = dev.get_macros()["u"].cpu().numpy().reshape(3, nz, 12 * 16)
    z = np.arange(nz)
    exact = g / (2 * nu) * (z + 0.5) * (nz - z - 0.5) + g / (8 * nu) * (16 * (tau - 0.5) ** 2 / 3 - 1)
    assert np.abs(u[0] - exact[:, None]).max() <= 1e-6 * exact.max()
    assert np.abs(u[1:]).max() <= 1e-9 * exact.max()      # round-off residue of the start-up transient (~1e-14)


def test_couette_closed_form_on_gpu(gpu):
    """Moving-wall bounce-back on the GPU path alone against Eq. 41: paper-sized 15^3 box,
    top wall U = 2e-2, Re = U N / nu = 10: the steady profile is linear, u_x = U (z + 1/2) / N, exactly."""
    N, U = 15, 2e-2
    nu = U * N / 10.0
    tau = 3 * nu + 0.5
    dev = gpu.LBM(N, N, N, "D3Q19", "BGK", precision=64, tau=(tau, tau), bc=(0, 0, 1), rho_init=(1.0, 1.0),
                  wall_u={(2, 1): (U, 0.0, 0.0)})
    dev.init_from_seed(0)
    dev.step(int(12 * N * N / nu))
    u = dev.get_macros()["u"].cpu().numpy().reshape(3, N, N * N)
    exact = U * (np.arange(N) + 0.5) / N
    assert np.abs(u[0] - exact[:, None]).max() <= 1e-9 * U
    assert np.abs(u[1:]).max() <= 1e-12


def test_cfg5_reduced_1000_steps_fp32(gpu):
    """configs[4] on a reduced 28x24x20 grid (the oracle runs ~0.5 MLUPS), fp32 against the fp32
    oracle, 1000 steps: fields <= 1e-5 (north_star); bit-exact by construction (psi = rho)."""
    cfg = workloads.config("cfg5", grid=(28, 24, 20), rmin=4.0, rmax=8.0, vol_frac=0.1)
    ref, dev = run_1000(gpu, cfg, 5)
    errs = macro_errs(ref, dev)
    assert max(errs.values()) <= 1e-5, errs
    assert np.array_equal(ref.get_populations(), dev.get_populations().cpu().numpy())


def tile_populations(f_small, nvals, small, full, device):
    """(nvals, nz, ny, nx) periodic tile of a small canonical population array to the full grid."""
    sx, sy, sz = small
    fx, fy, fz = full
    t = torch.from_numpy(f_small.reshape(nvals, sz, sy, sx)).to(device)
    return t.repeat(1, fz // sz, fy // sy, fx // sx).reshape(-1)


def check_tiled(out, ref_small, nvals, small, full):
    sx, sy, sz = small
    fx, fy, fz = full
    o = out.reshape(nvals, fz // sz, sz, fy // sy, sy, fx // sx, sx)
    r = torch.from_numpy(ref_small.reshape(nvals, 1, sz, 1, sy, 1, sx)).to(out.device)
    return bool((o == r).all().item())


@pytest.mark.parametrize("name,small,over,nsteps", [
    ("cfg3", (32, 16, 1), {}, 5),
    ("cfg4", (8, 4, 256), dict(init_kind="UNIFORM_NOISE", noise_amp=0.05), 5),
    ("cfg4", (8, 4, 256), dict(init_kind="UNIFORM_NOISE", noise_amp=0.05, precision=32), 4),
    ("cfg5", (16, 8, 8), dict(rmin=2.0, rmax=4.0, vol_frac=0.1), 3),
], ids=lambda v: str(v).replace(" ", ""))
def test_full_size_equals_tiled_small_oracle(gpu, name, small, over, nsteps):
    """Full BASELINE.json sizes (512^2, 256^3, 512^3) in the launch configuration bench.py times:
    a periodic tiling of a small seeded state stays a periodic tiling, so every cell of the full
    grid must equal, bit for bit, the oracle's result on the small grid."""
    from oracle.ref_lbm import RefLBM
    full = workloads.CONFIGS[name]["grid"]
    cs = workloads.config(name, grid=small, **over)
    cf = workloads.config(name, **over)
    ref = RefLBM(*cs["grid"], cs["lattice"], cs["model"], **cs["params"])
    ref.init_from_seed(11)
    nvals = ref.population_count() // ref.N
    dev = gpu.LBM(*cf["grid"], cf["lattice"], cf["model"], **cf["params"])
    big = tile_populations(ref.get_populations(), nvals, small, full, dev.device)
    dev.set_populations(big)
    del big
    ref.step(nsteps)
    dev.step(nsteps)
    out = dev.get_populations()
    assert check_tiled(out, ref.get_populations(), nvals, small, full)
    del out
    torch.cuda.empty_cache()


def test_cfg5_full_size_invariants(gpu):
    """configs[4] at 512^3 from its own seeded init: masses of A and B conserved, total C
    non-increasing and bounded below by C0 (1-k)^t (reaction sink, R8), no NaN."""
    cfg = workloads.config("cfg5")
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.init_from_seed(42)
    m = dev.get_macros(u=False, phi=False)
    m0 = m["rho"].double().sum(1).cpu().numpy()
    c0 = m["C"].double().sum().item()
    vol = (m["rho"][0] > 1.0).double().mean().item()
    assert 0.03 <= vol <= 0.07            # ~5 % volume fraction of component A (overlaps allowed)
    del m
    nsteps = 20
    dev.step(nsteps)
    m = dev.get_macros(phi=False)
    assert bool(torch.isfinite(m["u"]).all().item())
    m1 = m["rho"].double().sum(1).cpu().numpy()
    c1 = m["C"].double().sum().item()
    assert np.abs(m1 / m0 - 1).max() <= 1e-4        # fp32 populations, fp64 sum
    assert c0 * (1 - 1e-3) ** nsteps * (1 - 1e-5) <= c1 <= c0 * (1 + 1e-6)
    del m, dev
    torch.cuda.empty_cache()


def test_run_host_matches_device_path(gpu):
    """lbm_run_host (host buffers in and out, copies inside) gives the same bits as the device calls."""
    cfg = workloads.config("cfg4", grid=(16, 12, 10))
    ref, dev = make_pair(gpu, cfg)
    ref.init_from_seed(3)
    f0 = ref.get_populations()
    rho = np.empty((1, dev.N))
    u = np.empty((3, dev.N))
    dev.run_host(f0, 7, rho=rho, u=u)
    ref.step(7)
    mr = ref.get_macros()
    assert np.array_equal(rho, mr["rho"]) and np.array_equal(u, mr["u"])
    assert dev.time() == 7 and dev.launch_count() > 0


def test_errors_and_state(gpu):
    cfg = workloads.config("cfg1", grid=(8, 8, 1))
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    with pytest.raises(gpu.LbmError) as e:
        dev.step(1)                                   # before init
    assert e.value.code == -4
    dev.init_from_seed(0)
    dev.step(0)
    with pytest.raises(gpu.LbmError):
        dev.step(-1)
    buf = dev._new(dev.N)
    assert dev.L.lbm_get_macros(dev.h, None, None, None, buf.data_ptr()) == -1   # BGK has no scalar lattice
    assert "scalar" in gpu.lbm.last_error()
    with pytest.raises(gpu.LbmError):
        gpu.LBM(8, 8, 2, "D2Q9", "BGK")               # D2Q9 needs nz == 1
    sc = gpu.LBM(8, 8, 1, "D2Q9", "SC1", bc=(1, 0, 0))
    with pytest.raises(gpu.LbmError):
        sc.set_path("pipeline")                       # walls in x: register path only


PATH_CASES = [
    ("cfg2", (300, 21, 1), dict(radius=6.0)),
    ("cfg2", (256, 40, 1), dict(radius=9.0)),
    ("cfg3", (260, 37, 1), {}),
    ("cfg3", (132, 5, 1), dict(precision=32)),
    ("cfg3", (8, 3, 1), {}),
    ("cfg5", (140, 9, 7), dict(rmin=2.0, rmax=4.0, vol_frac=0.1)),
    ("cfg5", (264, 12, 10), dict(rmin=2.0, rmax=4.0, vol_frac=0.1)),
    ("cfg5", (16, 3, 2), dict(rmin=1.0, rmax=2.0, vol_frac=0.1)),
    ("cfg5", (8, 1, 1), dict(rmin=1.0, rmax=2.0, vol_frac=0.1)),
    ("cfg5", (4, 2, 3), dict(rmin=1.0, rmax=2.0, vol_frac=0.1)),
    ("cfg5", (136, 6, 5), dict(rmin=2.0, rmax=3.0, vol_frac=0.1, precision=64, tau=(0.9, 1.1), tau_c=0.7)),
    ("cfg5", (12, 9, 7), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, force=(1e-5, -2e-5, 3e-5), tau=(0.8, 1.3))),
    # walls in y / z (uniform per row): halfway bounce-back, fluid-only stencil, adhesion (Eq. 11-12, 14)
    ("cfg2", (136, 17, 1), dict(radius=5.0, bc=(0, 1, 0), G_ads=(-0.4, 0.0))),
    ("cfg2", (20, 12, 1), dict(radius=4.0, bc=(0, 1, 0), rho_wall=1.2)),
    ("cfg3", (16, 9, 1), dict(bc=(0, 1, 0), G_ads=(-0.2, 0.3), force=(1e-5, -2e-5, 0.0))),
    ("cfg5", (12, 9, 7), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, bc=(0, 0, 1), G_ads=(-0.3, 0.3))),
    ("cfg5", (132, 6, 5), dict(rmin=1.0, rmax=2.0, vol_frac=0.2, bc=(0, 1, 1), G_ads=(0.1, -0.2))),
    ("cfg5", (8, 6, 5), dict(rmin=1.0, rmax=2.0, vol_frac=0.2, bc=(0, 1, 1), G_ads=(0.1, -0.2), precision=64, tau=(0.9, 1.1))),
    # moving walls in y / z (sheared two-component flow)
    ("cfg5", (264, 9, 7), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, bc=(0, 1, 1), G_ads=(-0.3, 0.3), tau=(0.9, 1.2),
                              wall_u={(2, 1): (0.02, -0.01, 0.0), (2, 0): (-0.02, 0.0, 0.0), (1, 0): (0.01, 0.0, 0.02)})),
    ("cfg3", (132, 9, 1), dict(bc=(0, 1, 0), G_ads=(-0.2, 0.3), wall_u={(1, 0): (0.01, 0.0, 0.0), (1, 1): (-0.02, 0.0, 0.0)})),
    ("cfg2", (136, 12, 1), dict(radius=4.0, bc=(0, 1, 0), G_ads=(-0.3, 0.0), wall_u={(1, 1): (0.02, 0.0, 0.0)})),
    # velocity-shift forcing scheme (forcing = 1, Eq. 16-19) with unequal relaxation times
    ("cfg5", (264, 12, 10), dict(forcing=1, rmin=2.0, rmax=4.0, vol_frac=0.1, tau=(0.9, 1.2))),
    ("cfg5", (12, 9, 7), dict(forcing=1, rmin=2.0, rmax=3.0, vol_frac=0.2, precision=64, tau=(0.9, 1.1), tau_c=0.7, bc=(0, 1, 0), G_ads=(0.2, -0.1))),
    ("cfg3", (260, 37, 1), dict(forcing=1, force=(1e-5, 2e-5, 0.0), tau=(0.8, 1.3))),
    ("cfg3", (132, 5, 1), dict(forcing=1, precision=32, bc=(0, 1, 0), G_ads=(0.25, -0.25))),
    ("cfg2", (256, 40, 1), dict(forcing=1, radius=9.0)),
]
PATHS = [("register", 0), ("pipeline", 0), ("pipeline", 1), ("pipeline", 3), ("pipeline", 1000)]


@pytest.mark.parametrize("name,grid,over", PATH_CASES, ids=lambda v: str(v).replace(" ", ""))
@pytest.mark.parametrize("path", PATHS, ids=lambda v: "%s-%d" % v)
def test_every_path_matches_oracle(gpu, name, grid, over, path):
    """Both launch paths of lbm_step (include/lbm.h LBM_PATH_*: register kernels; the persistent resident-tile
    kernel) with several schedules (pencils of 1 / 3 / all rows) against the oracle at every step 1..7, on rows
    of several tiles with a ragged tail, on degenerate extents, with walls in y / z, fp64 and fp32 (packed)."""
    cfg = workloads.config(name, grid=grid, **over)
    ref, dev = make_pair(gpu, cfg)
    dev.set_path(*path)
    assert dev.get_path() == path[0]
    ref.init_from_seed(9)
    dev.set_populations(torch.from_numpy(ref.get_populations()))
    exact = not (cfg["model"] == "SC1" and cfg["params"].get("psi_kind", 0) == 0)
    for step in range(1, 8):
        ref.step(1)
        dev.step(1)
        fr = ref.get_populations()
        fd = dev.get_populations().cpu().numpy()
        if exact:
            assert np.array_equal(fr, fd), "step %d: %d of %d differ" % (step, (fr != fd).sum(), fr.size)
        else:
            assert np.abs(fr - fd).max() <= 1e-13 * np.abs(fr).max(), "step %d" % step
    dev.check()
    assert dev.launch_count() >= 7


def test_pipeline_path_rejects_what_it_does_not_handle(gpu):
    cfg = workloads.config("cfg3", grid=(9, 4, 1))
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    with pytest.raises(gpu.LbmError):
        dev.set_path("pipeline")                     # 9 doubles per row: rows are not 16-byte aligned
    assert dev.get_path() == "register"
    cfg = workloads.config("cfg3", grid=(8, 4, 1), bc=(1, 0, 0))
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    with pytest.raises(gpu.LbmError):
        dev.set_path("pipeline")                     # walls in x
    cfg = workloads.config("cfg3", grid=(8, 4, 1), forcing=1)
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.set_path("pipeline")                         # velocity-shift forcing: handled
    assert dev.get_path() == "pipeline"
    cfg = workloads.config("cfg4", grid=(8, 4, 4))
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    with pytest.raises(gpu.LbmError):
        dev.set_path("pipeline")                     # BGK: the register path already moves the algorithmic bytes
    with pytest.raises(gpu.LbmError):
        gpu.LBM(8, 4, 1, "D2Q9", "SC2", bc=(0, 1, 0), forcing=1, wall_u={(1, 1): (0.01, 0.0, 0.0)})   # moving walls need Guo forcing


def test_default_path_of_large_shan_chen_grids(gpu):
    """Without lbm_set_path a two-component D3Q19 fp32 context with more than 2^21 cells switches to the resident-tile
    path at its first step (include/lbm.h); the result equals the register path bit for bit.  D2Q9 fp64 contexts
    stay on the register kernels (measured faster there)."""
    cfg = workloads.config("cfg5", grid=(512, 96, 48), rmin=4.0, rmax=8.0)
    a = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    b = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    b.set_path("register")
    a.init_from_seed(3)
    b.init_from_seed(3)
    a.step(5)
    b.step(5)
    assert a.get_path() == "pipeline" and b.get_path() == "register"
    assert torch.equal(a.get_populations(), b.get_populations())
    ma, mb = a.get_macros(), b.get_macros()
    for k in ma:
        assert torch.equal(ma[k], mb[k]), k
    a.check()
    cfg = workloads.config("cfg3", grid=(2048, 1032, 1))
    c = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    c.init_from_seed(3)
    c.step(2)
    assert c.get_path() == "register"


@pytest.mark.parametrize("name,grid,over", [
    ("cfg5", (520, 72, 48), dict(rmin=4.0, rmax=8.0, bc=(0, 1, 1), G_ads=(-0.2, 0.3))),       # ragged x tiles, walls in y and z
    ("cfg5", (1024, 40, 36), dict(rmin=4.0, rmax=8.0, force=(1e-6, -2e-6, 3e-6))),             # four tiles per row
    ("cfg5", (512, 64, 40), dict(rmin=4.0, rmax=8.0, forcing=1, tau=(0.9, 1.2))),                # velocity-shift forcing
    ("cfg5", (512, 48, 40), dict(rmin=4.0, rmax=8.0, bc=(0, 0, 1), wall_u={(2, 0): (-0.02, 0.0, 0.0), (2, 1): (0.02, 0.01, 0.0)})),   # shear
    ("cfg3", (4096, 300, 1), dict(bc=(0, 1, 0), G_ads=(0.1, -0.1))),                           # D2Q9 fp64, walls in y
    ("cfg2", (2048, 260, 1), dict(radius=60.0)),                                                # D2Q9 SC1 fp64 (psi with exp)
], ids=lambda v: str(v).replace(" ", ""))
def test_tile_path_equals_register_path_with_many_tickets_per_block(gpu, name, grid, over):
    """The resident-tile kernel with every block working through many tickets (thousands of tiles on 148 blocks, psi parts
    waiting on flags of other blocks, ragged tiles at the end of a row, walls in y / z), against the register kernels on
    the same seeded input after 7 steps (both AA parities): bit for bit -- both paths run the same per-cell device code,
    and the register path is compared with the oracle everywhere else in this file."""
    cfg = workloads.config(name, grid=grid, **over)
    a = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    b = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    a.set_path("pipeline")
    b.set_path("register")
    a.init_from_seed(5)
    b.init_from_seed(5)
    for n in (1, 2, 4):
        a.step(n)
        b.step(n)
        fa, fb = a.get_populations(), b.get_populations()
        assert torch.equal(fa, fb), "after %d steps: %d populations differ" % (a.time(), int((fa != fb).sum().item()))
        del fa, fb
    ma, mb = a.get_macros(), b.get_macros()
    for k in ma:
        if ma[k] is not None:
            assert torch.equal(ma[k], mb[k]), k
    a.check()
    a.close()
    b.close()
    torch.cuda.empty_cache()


MASK_CASES = [
    ("cfg1", (20, 13, 1), dict(force=(1e-5, 2e-5, 0.0))),
    ("cfg1", (132, 9, 1), {}),
    ("cfg4", (9, 8, 7), dict(bc=(0, 0, 1))),
    ("cfg4", (12, 6, 5), dict(bc=(0, 0, 0), precision=32)),
    ("cfg4", (7, 6, 5), dict(bc=(0, 0, 1), force=(0.0, 0.0, 0.0), wall_u={(2, 1): (0.02, 0.0, 0.0)})),
    ("cfg2", (16, 12, 1), dict(radius=4.0, G_ads=(-0.3, 0.0))),
    ("cfgT", (9, 8, 6), {}),
    # solid-phase internal-energy lattice on the solid nodes (Eq. 31-33), walls in z / fully periodic / 2D fp32
    ("cfgT", (9, 8, 6), dict(tau_s=0.9, rho_solid=2.0)),
    ("cfgT", (7, 6, 5), dict(tau_s=1.4, rho_solid=0.5, bc=(0, 0, 0), force=(0.0, 0.0, 0.0))),
    ("cfgT2", (13, 11, 1), dict(tau_s=0.75, rho_solid=1.5, precision=32)),
    # Eq. 12 solid term next to solid nodes of the mask (and next to walls as well)
    ("cfg2", (16, 12, 1), dict(radius=4.0, rho_wall=1.5)),
    ("cfg2", (14, 10, 1), dict(radius=3.0, rho_wall=0.4, G_ads=(-0.2, 0.0), bc=(0, 1, 0))),
    ("cfg3", (14, 11, 1), dict(G_ads=(-0.2, 0.3))),
    ("cfg5", (10, 8, 6), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, G_ads=(0.2, -0.2))),
    ("cfg5", (8, 7, 6), dict(rmin=2.0, rmax=3.0, vol_frac=0.2, forcing=1, bc=(0, 1, 0), precision=64, tau=(0.9, 1.2))),
]


@pytest.mark.parametrize("name,grid,over", MASK_CASES, ids=lambda v: str(v).replace(" ", ""))
def test_solid_mask_matches_oracle(gpu, name, grid, over):
    """lbm_set_mask: a random 15 % of the nodes solid (isolated nodes, clusters, nodes next to walls and across the
    periodic seam): populations at every step 1..12 (odd and even AA parity), macros and forces against the oracle."""
    cfg = workloads.config(name, grid=grid, **over)
    ref, dev = make_pair(gpu, cfg)
    mask = (np.random.default_rng(1).random(ref.N) < 0.15).astype(np.uint8)
    ref.init_from_seed(3)
    dev.set_populations(torch.from_numpy(ref.get_populations()))
    ref.set_mask(mask)
    dev.set_mask(mask)
    exact = not (cfg["model"] == "SC1" and cfg["params"].get("psi_kind", 0) == 0)
    for step in range(1, 13):
        ref.step(1)
        dev.step(1)
        fr = ref.get_populations()
        fd = dev.get_populations().cpu().numpy()
        if exact:
            assert np.array_equal(fr, fd), "step %d" % step
        else:
            assert np.abs(fr - fd).max() <= 1e-13 * np.abs(fr).max(), "step %d" % step
        if step == 11:
            with pytest.raises(gpu.LbmError):
                dev.set_mask(None)                 # odd time level: the layout depends on the mask
    mr, md = ref.get_macros(), dev.get_macros()
    tol = 0.0 if exact else 1e-13
    assert field_err(md["rho"].cpu().numpy(), mr["rho"]) <= tol
    assert field_err(md["u"].cpu().numpy(), mr["u"]) <= tol
    if mr["C"] is not None:                        # scalar / internal energy, eps_s on solid nodes that carry a lattice
        assert field_err(md["C"].cpu().numpy(), mr["C"]) <= tol
        if cfg["params"].get("tau_s", 0.0) > 0.0:
            assert np.all(mr["C"][mask != 0] > 0.0)
    solid = mask != 0
    assert not md["rho"].cpu().numpy()[:, solid].any() and not md["u"].cpu().numpy()[:, solid].any()
    Fr, Fd = ref.get_force(), dev.get_force().cpu().numpy()
    assert np.abs(Fr - Fd).max() <= tol * max(np.abs(Fr).max(), 1e-300)
    # clearing the mask returns to the plain kernels
    dev.set_mask(None)
    ref.set_mask(None)
    ref.step(2)
    dev.step(2)
    if exact:
        assert np.array_equal(ref.get_populations(), dev.get_populations().cpu().numpy())
    with pytest.raises(gpu.LbmError):
        dev.set_mask(mask)
        dev.set_path("pipeline")                 # a masked context runs on the register path


def test_masked_graph_replay_and_mass(gpu):
    """Flow past an obstacle over 200 steps (CUDA-graph replay on a small grid, rebuilt after lbm_set_mask):
    equals the oracle bit for bit; mass of the fluid nodes conserved."""
    nx, ny = 24, 17
    cfg = workloads.config("cfg1", grid=(nx, ny, 1), init_kind="REST", force=(1e-6, 0.0, 0.0))
    ref, dev = make_pair(gpu, cfg)
    m = np.zeros((ny, nx), np.uint8)
    m[6:11, 8:13] = 1
    ref.init_from_seed(0)
    dev.init_from_seed(0)
    dev.step(40)                              # builds the graph without a mask
    ref.step(40)
    ref.set_mask(m)
    dev.set_mask(m)
    ref.step(200)
    dev.step(200)
    fr, fd = ref.get_populations(), dev.get_populations().cpu().numpy()
    assert np.array_equal(fr, fd)
    fluid = np.tile(m.ravel() == 0, 9)
    assert abs(fd[fluid].sum() - (m == 0).sum()) < 1e-9


# ------------------------------------------------------------------------------------------------------
# the BASELINE.json configurations at their full sizes and step counts, checked by what the method fixes
# (closed forms and invariants; R15: field parity with the oracle is at 1000 steps, see above)
# ------------------------------------------------------------------------------------------------------
def test_cfg2_laplace_law_full_run(gpu):
    """configs[1] as stated: 256x256, R in {20, 30, 40, 50}, 20000 steps each: the pressure jump of the relaxed
    droplet, p = rho/3 + (G/6) psi^2, times the MEASURED radius is the same constant for every droplet
    (Laplace law dp = gamma / R: PAPER.md:636-676); mass conserved to round-off."""
    res = []
    for R in (20.0, 30.0, 40.0, 50.0):
        cfg = workloads.config("cfg2", radius=R)
        dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
        dev.init_from_seed(2)
        m0 = dev.get_macros(u=False, phi=False)["rho"].sum().item()
        dev.step(20000)
        mac = dev.get_macros(phi=False)
        rho = mac["rho"][0].cpu().numpy().reshape(256, 256)
        assert abs(rho.sum() / m0 - 1) < 1e-10
        psi = 1 - np.exp(-rho)
        p = rho / 3 + (-5.0 / 6) * psi ** 2
        rin, rout = rho[128, 128], rho[0, 0]
        assert rin > 1.8 and rout < 0.2
        reff = np.sqrt(((rho - rout) / (rin - rout)).sum() / np.pi)
        res.append((1 / reff, p[128, 128] - p[0, 0]))
        assert mac["u"].abs().max().item() < 0.02
    inv_r, dp = np.array(res).T
    gamma = dp / inv_r
    assert (dp > 0).all() and (np.diff(dp) < 0).all()
    assert gamma[1:].max() / gamma[1:].min() - 1 < 0.03        # the three larger droplets
    assert gamma.max() / gamma.min() - 1 < 0.10                # all four (the smallest shrinks to R_eff ~ 8)


def test_cfg3_full_run_mass_and_demixing(gpu):
    """configs[2] as stated: 512x512, 10000 steps of spinodal decomposition: per-component mass conserved to
    round-off, the mixture has separated into A-rich and B-rich domains, everything finite."""
    cfg = workloads.config("cfg3")
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.init_from_seed(3)
    m0 = dev.get_macros(u=False, phi=False)["rho"].sum(1).cpu().numpy()
    dev.step(10000)
    mac = dev.get_macros()
    m1 = mac["rho"].sum(1).cpu().numpy()
    assert np.abs(m1 / m0 - 1).max() < 1e-10
    phi = mac["phi"].cpu().numpy()
    assert np.isfinite(phi).all() and bool(torch.isfinite(mac["u"]).all().item())
    assert (phi > 0.5).mean() > 0.2 and (phi < -0.5).mean() > 0.2       # two phases, each a sizeable share of the box
    assert abs(phi.mean()) < 0.05                                        # symmetric mixture


# measured on the B200 (this test prints it): see DESIGN.md R13
DRIFT_BOUND_CFG5 = 1e-4     # measured 3.3e-5 (A), 3.1e-5 (B) relative drift after 2000 fp32 steps: 3 x that = SURVEY 8(c)'s 1e-4


def test_cfg5_full_run_invariants(gpu):
    """configs[4] as stated: 512^3, fp32, 2000 steps: masses of A and B conserved (fp32 populations, fp64 sums),
    total C decreasing and bounded below by C0 (1 - k)^t (the reaction factor 4 rhoA rhoB / rho^2 is <= 1), no NaN."""
    cfg = workloads.config("cfg5")
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.init_from_seed(42)
    m = dev.get_macros(u=False, phi=False)
    m0 = m["rho"].double().sum(1).cpu().numpy()
    c0 = m["C"].double().sum().item()
    del m
    dev.step(2000)
    m = dev.get_macros(phi=False)
    assert bool(torch.isfinite(m["u"]).all().item()) and bool(torch.isfinite(m["rho"]).all().item())
    m1 = m["rho"].double().sum(1).cpu().numpy()
    c1 = m["C"].double().sum().item()
    drift = np.abs(m1 / m0 - 1).max()
    print("cfg5 512^3 fp32, 2000 steps: relative mass drift per component", (m1 / m0 - 1).tolist())
    assert drift <= DRIFT_BOUND_CFG5
    assert c0 * (1 - 1e-3) ** 2000 * (1 - 1e-4) <= c1 < c0
    del m, dev
    torch.cuda.empty_cache()


def test_contact_angle_versus_adhesion(gpu):
    """Wettability: a half droplet of component 1 on the wall y = -1/2 in component 2, D2Q9 two
    components with psi = rho, cohesion G_c, adhesion G_ads,1 = -G_ads,2 (Eq. 14).  The contact angle is measured as the
    paper does, from the height h and the contact length b of the region where component 1 dominates (Eq. 49-50), for
    dG = G_ads,2 - G_ads,1 in {-0.4, -0.2, 0, 0.2, 0.4}.  What the method fixes and this test asserts: a neutral wall gives
    90 degrees; cos(theta) is odd and LINEAR in dG (Eq. 48: cos(theta) = dG / (G_c (rho_1 - rho_2) / 2)).  The measured
    slope is 1.9 times the slope Eq. 48 prints (R26 records the discrepancy and bounds it here)."""
    nx, ny, Gc, rho_m, rho_d, R0 = 200, 100, 1.5, 2.0, 0.06, 30.0
    c, w, _ = gpu.lbm.lattice_table("D2Q9")
    y, x = np.mgrid[0:ny, 0:nx]
    d = np.sqrt((x - (nx - 1) / 2) ** 2 + (y + 0.5) ** 2)          # centre on the wall
    ind = 0.5 * (1 - np.tanh(2 * (d - R0) / 4.0))
    rA, rB = rho_d + (rho_m - rho_d) * ind, rho_m - (rho_m - rho_d) * ind
    f0 = np.concatenate([(w[:, None] * rA.ravel()[None, :]).ravel(), (w[:, None] * rB.ravel()[None, :]).ravel()])

    def cos_theta(dG):
        sim = gpu.LBM(nx, ny, 1, "D2Q9", "SC2", precision=64, tau=(1.0, 1.0), psi_kind=1, G=((0.0, Gc), (Gc, 0.0)),
                      bc=(0, 1, 0), G_ads=(-dG / 2.0, dG / 2.0))
        sim.set_populations(torch.from_numpy(f0))
        sim.step(16000)
        rho = sim.get_macros(u=False, phi=False)["rho"].cpu().numpy().reshape(2, ny, nx)
        sim.close()
        phi = rho[0] - rho[1]
        col = phi[:, nx // 2]
        j = np.where(col > 0)[0].max()
        h = (j + 0.5) + col[j] / (col[j] - col[j + 1])               # height above the wall (cell centres at y = j)
        row = 1.5 * phi[0] - 0.5 * phi[1]                              # phi extrapolated to the wall
        k = np.where(row > 0)[0]
        b = (k.max() + row[k.max()] / (row[k.max()] - row[k.max() + 1])) - (k.min() - row[k.min()] / (row[k.min()] - row[k.min() - 1]))
        r = (4 * h * h + b * b) / (8 * h)                              # Eq. 49
        theta = np.pi - np.arctan(b / (2 * (h - r))) if h > r else np.arctan(b / (2 * (r - h)))     # Eq. 50 and its lower branch
        inside = rho[0] > rho[1]
        return np.cos(theta), rho[0][inside].max(), rho[0][ny - 5, 5]

    res = {dG: cos_theta(dG) for dG in (-0.4, -0.2, 0.0, 0.2, 0.4)}
    cs = {k: v[0] for k, v in res.items()}
    print("contact angle: cos(theta) by dG", cs)
    assert abs(cs[0.0]) < 0.05                                         # neutral wall: 90 degrees
    assert abs(cs[0.2] + cs[-0.2]) < 0.06 and abs(cs[0.4] + cs[-0.4]) < 0.06          # odd in dG
    assert cs[-0.4] < cs[-0.2] < cs[0.0] < cs[0.2] < cs[0.4]           # G_ads,1 < 0: component 1 wets the wall more
    assert abs(cs[0.4] / cs[0.2] - 2.0) < 0.15 and abs(cs[-0.4] / cs[-0.2] - 2.0) < 0.15   # linear
    slope = (cs[0.4] - cs[-0.4]) / 0.8
    rho1, rho2 = res[0.0][1], res[0.0][2]
    slope48 = 1.0 / (Gc * (rho1 - rho2) / 2.0)                         # Eq. 48
    print("slope %.3f, Eq. 48 slope %.3f, ratio %.2f" % (slope, slope48, slope / slope48))
    assert 1.6 < slope / slope48 < 2.2


@pytest.mark.skipif(not __import__("os").environ.get("LBM_LONG"), reason="9 min on a B200: set LBM_LONG=1")
def test_cfg4_full_size_steady_state(gpu):
    """configs[3] 'run to steady state' at the full 256^3 (700 000 steps, fp64): the Poiseuille profile with the
    halfway-bounce-back slip term, u_x(z) = g/(2 nu) (z+1/2)(H-z-1/2) + g/(8 nu) (16 (tau-1/2)^2/3 - 1)."""
    cfg = workloads.config("cfg4")
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.init_from_seed(0)
    for _ in range(70):
        dev.step(10000)
        dev.synchronize()
    nz, tau, g = 256, 0.9, 1e-6
    nu = (tau - 0.5) / 3
    u = dev.get_macros(phi=False)["u"].reshape(3, nz, -1)
    z = np.arange(nz)
    exact = g / (2 * nu) * (z + 0.5) * (nz - z - 0.5) + g / (8 * nu) * (16 * (tau - 0.5) ** 2 / 3 - 1)
    ux = u[0].cpu().numpy()
    err = np.abs(ux - exact[:, None]).max() / exact.max()
    print("cfg4 256^3 steady state: max |u_x - exact| / u_max = %.3e" % err)
    assert err < 1e-5
    assert u[1:].abs().max().item() < 1e-9 * exact.max()
