"""lbm_step_static (include/lbm.h): the Shan-Chen step without any allocation -- the psi field lives in a static device
array of the library -- against the existing path (lbm_create / lbm_set_populations / lbm_step / lbm_get_populations).
`-m gpu`.  Collected last on purpose (the suite runs with pytest -x).

Both sides run the same register kernels on the same inputs, so the populations must agree BIT FOR BIT (the bar the
parity tests use for GPU-vs-oracle on the models without a transcendental; here it also holds for psi = 1 - exp(-rho),
because both sides call the same device code).  Two calls in a row with different shapes and precisions share the scratch
array: the second must not be affected by what the first left there.
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
    ge.build()
    import paper_2502_12955_b200 as lbm
    lbm.lib()
    return lbm


CASES = [
    # (config, grid, overrides, steps)
    ("cfg5", (40, 24, 20), dict(rmin=3.0, rmax=5.0, vol_frac=0.1), 6),                       # D3Q19 SC2 + D3Q7, fp32
    ("cfg3", (96, 50, 1), dict(bc=(0, 1, 0), G_ads=(-0.2, 0.3), force=(1e-5, -2e-5, 0.0)), 8),   # D2Q9 SC2 fp64, walls
    ("cfg2", (64, 40, 1), dict(radius=10.0), 4),                                               # D2Q9 SC1 fp64, psi with exp
    ("cfg5", (40, 24, 20), dict(rmin=3.0, rmax=5.0, vol_frac=0.1), 6),                       # the first case again
]


def reference_run(gpu, cfg, steps):
    """(canonical populations at t = 0, at t = steps) from the existing path"""
    dev = gpu.LBM(*cfg["grid"], cfg["lattice"], cfg["model"], **cfg["params"])
    dev.set_path("register")
    dev.init_from_seed(11)
    f0 = dev.get_populations().clone()
    dev.step(steps)
    f1 = dev.get_populations().clone()
    dev.close()
    return f0, f1


def test_step_static_matches_the_existing_path_on_calls_in_a_row(gpu):
    prepared = []
    for name, grid, over, steps in CASES:
        cfg = workloads.config(name, grid=grid, **over)
        f0, f1 = reference_run(gpu, cfg, steps)
        prepared.append((cfg, steps, f0.clone(), f1))
    torch.cuda.synchronize()
    for k, (cfg, steps, f, expect) in enumerate(prepared):          # calls in a row, nothing else in between
        gpu.lbm.step_static(*cfg["grid"], cfg["lattice"], cfg["model"], f, steps, **cfg["params"])
    torch.cuda.synchronize()
    for k, (cfg, steps, f, expect) in enumerate(prepared):
        bad = int((f != expect).sum().item())
        assert bad == 0, "call %d (%s %s): %d of %d populations differ from lbm_step" % (k, cfg["lattice"], cfg["model"], bad, f.numel())
        assert bool(torch.isfinite(f).all().item())


def test_step_static_allocates_nothing_and_checks_its_limits(gpu):
    name, grid, over, steps = CASES[0]
    cfg = workloads.config(name, grid=grid, **over)
    f0, f1 = reference_run(gpu, cfg, steps)
    fa, fb = f0.clone(), f0.clone()
    gpu.lbm.step_static(*cfg["grid"], cfg["lattice"], cfg["model"], fa, steps, **cfg["params"])     # (loads the kernels)
    torch.cuda.synchronize()
    unchanged = False
    for attempt in range(3):        # (device-wide figure: repeat if something else on the box moved it)
        fb.copy_(f0)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        gpu.lbm.step_static(*cfg["grid"], cfg["lattice"], cfg["model"], fb, steps, **cfg["params"])
        torch.cuda.synchronize()
        if torch.cuda.mem_get_info()[0] == free_before:
            unchanged = True
            break
    assert unchanged                                            # no device memory was taken
    assert torch.equal(fa, f1) and torch.equal(fb, f1)
    # n = 0 leaves the array alone
    fc = f0.clone()
    gpu.lbm.step_static(*cfg["grid"], cfg["lattice"], cfg["model"], fc, 0, **cfg["params"])
    torch.cuda.synchronize()
    assert torch.equal(fc, f0)
    # limits: the psi field must fit the static array; even n; Shan-Chen models only
    cap = gpu.lbm.static_scratch_bytes()
    assert cap == 16 << 20
    big = workloads.config("cfg5", grid=(256, 128, 128))           # 2 * 2^22 cells * 4 bytes = 32 MiB of psi
    dummy = torch.zeros(16, dtype=torch.float32, device="cuda")
    with pytest.raises(gpu.LbmError) as e:
        gpu.lbm.step_static(*big["grid"], big["lattice"], big["model"], dummy, 2, **big["params"])
    assert e.value.code == -1 and "static scratch holds" in str(e.value)
    fits = workloads.config("cfg5", grid=(128, 128, 128))          # exactly 16 MiB: accepted (n = 0: nothing is touched)
    gpu.lbm.step_static(*fits["grid"], fits["lattice"], fits["model"], dummy, 0, **fits["params"])
    with pytest.raises(gpu.LbmError):
        gpu.lbm.step_static(*cfg["grid"], cfg["lattice"], cfg["model"], fc, 3, **cfg["params"])       # odd n
    bgk = workloads.config("cfg4", grid=(16, 8, 8))
    with pytest.raises(gpu.LbmError):
        gpu.lbm.step_static(*bgk["grid"], bgk["lattice"], bgk["model"], dummy, 2, **bgk["params"])    # no psi field
