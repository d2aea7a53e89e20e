"""The five BASELINE.json configurations (and reduced parity-test variants) as plain parameter
dictionaries.  Inputs only: this module holds none of the method's arithmetic and imports neither
the oracle nor the CUDA library; both bindings accept these keyword arguments.

Readings of the paper behind each value: DESIGN.md "Readings" (R-numbers) and "Input recipe".
"""

G12 = ((0.0, 1.2), (1.2, 0.0))  # inter-component coupling only, no self-interaction (configs 3, 5)

CONFIGS = {
    # config 1: D2Q9 BGK, Taylor-Green vortex, closed-form decay (BASELINE.json configs[0])
    "cfg1": dict(grid=(64, 64, 1), lattice="D2Q9", model="BGK", steps=1000,
                 params=dict(precision=64, tau=(0.8, 0.8), rho_init=(1.0, 1.0), u0=0.01,
                             init_kind="TAYLOR_GREEN")),
    # config 2: D2Q9 single-component Shan-Chen droplet, Laplace law (configs[1]); radius swept by the caller
    "cfg2": dict(grid=(256, 256, 1), lattice="D2Q9", model="SC1", steps=20000,
                 params=dict(precision=64, tau=(1.0, 1.0), psi_kind=0, rho0_psi=1.0,
                             G=((-5.0, 0.0), (0.0, 0.0)), init_kind="DROPLET", rho_in=2.0, rho_out=0.1,
                             radius=30.0, width=3.0, noise_amp=0.01)),
    # config 3: D2Q9 two-component Shan-Chen spinodal decomposition (configs[2]); psi = rho (R3)
    "cfg3": dict(grid=(512, 512, 1), lattice="D2Q9", model="SC2", steps=10000,
                 params=dict(precision=64, tau=(1.0, 1.0), psi_kind=1, G=G12, init_kind="UNIFORM_NOISE",
                             rho_init=(1.0, 1.0), noise_amp=0.01)),
    # config 4: D3Q19 BGK + Guo body force, halfway bounce-back walls in z (configs[3]); fp64 and fp32
    "cfg4": dict(grid=(256, 256, 256), lattice="D3Q19", model="BGK", steps=1000,
                 params=dict(precision=64, tau=(0.9, 0.9), force=(1e-6, 0.0, 0.0), bc=(0, 0, 1),
                             init_kind="REST", rho_init=(1.0, 1.0))),
    # config 5: D3Q19 two-component Shan-Chen + D3Q7 scalar with first-order interface reaction (configs[4])
    "cfg5": dict(grid=(512, 512, 512), lattice="D3Q19", model="SC2_ADE", steps=2000,
                 params=dict(precision=32, tau=(1.0, 1.0), tau_c=0.8, psi_kind=1, G=G12, k_react=1e-3,
                             init_kind="RANDOM_DROPLETS", rho_in=1.9, rho_out=0.1, c_init=1.0, width=3.0,
                             rmin=10.0, rmax=30.0, vol_frac=0.05)),
    # beyond BASELINE.json: BGK + internal-energy lattice (IEDDF, Eq. 27-30), 3D channel / 2D box
    "cfgT": dict(grid=(64, 64, 64), lattice="D3Q19", model="BGK_T", steps=1000,
                 params=dict(precision=64, tau=(0.9, 0.9), tau_c=0.8, force=(1e-6, 0.0, 0.0), bc=(0, 0, 1),
                             init_kind="TAYLOR_GREEN", u0=0.02, rho_init=(1.0, 1.0), c_init=0.5)),
    "cfgT2": dict(grid=(128, 128, 1), lattice="D2Q9", model="BGK_T", steps=1000,
                  params=dict(precision=64, tau=(0.8, 0.8), tau_c=0.7, init_kind="TAYLOR_GREEN", u0=0.03,
                              rho_init=(1.0, 1.0), c_init=1.5)),
}


def config(name, grid=None, **overrides):
    """A copy of CONFIGS[name] with an optional reduced grid and parameter overrides."""
    c = CONFIGS[name]
    out = dict(grid=tuple(grid) if grid is not None else c["grid"], lattice=c["lattice"], model=c["model"],
               steps=c["steps"], params=dict(c["params"]))
    out["params"].update(overrides)
    return out
