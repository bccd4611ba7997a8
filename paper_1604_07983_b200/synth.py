"""Seeded synthetic quark propagators (shared by the oracle tests and the CUDA path).

This module holds NONE of the method's arithmetic: it only draws the inputs.  It is the one
module both `oracle/` tests and the CUDA binding's callers may import ("Input recipe").

Recipe (BASELINE.json `configs`, reading A17): for every flavour f, time
slice t and site x the propagator S_f(x) is a 12x12 complex128 matrix [sink xi][source xi'],
xi = colour + 3*spin, whose real and imaginary parts are i.i.d. N(0,1), multiplied by
exp(-m_f * t).  The paper's real inputs (propagators on CP-PACS/JLQCD gauge configurations,
PAPER.md:147) are not available; these stand in for them.

The generator is counter-based (numpy Philox) keyed by (seed, stream, t), so any slice of any
flavour can be drawn without drawing the others.  `stream` separates flavours that share a seed.
"""
from __future__ import annotations

import numpy as np

NCS = 12  # colour x spin


def propagator(seed: int, stream: int, t: int, L: int, mass: float) -> np.ndarray:
    """One flavour on one time slice: array [L^3][12][12] complex128, site = x + L*(y + L*z)."""
    V = L * L * L
    bitgen = np.random.Philox(key=[int(seed) & (2**64 - 1), (int(stream) << 32) | int(t)])
    rng = np.random.Generator(bitgen)
    z = rng.standard_normal((V, NCS, NCS, 2))
    S = (z[..., 0] + 1j * z[..., 1]) * np.exp(-float(mass) * t)
    return np.ascontiguousarray(S, dtype=np.complex128)


# The five workloads of BASELINE.json `configs` (index = position in that list).
CONFIGS = [
    dict(name="cfg0_4c1_NN", L=4, T=1, channels="NN", flavours=dict(u=(0, 0, 0.2), d="u", s=(0, 1, 0.3))),
    dict(name="cfg1_16c32", L=16, T=32, channels="all52", flavours=dict(u=(1, 0, 0.2), d="u", s=(2, 0, 0.3))),
    dict(name="cfg2_32c64", L=32, T=64, channels="all52",
         flavours=dict(u=(3, 0, 0.20), d=(3, 1, 0.21), s=(3, 2, 0.30))),
    dict(name="cfg3_32c64_su3", L=32, T=64, channels="all52", flavours=dict(u=(4, 0, 0.25), d="u", s="u")),
    dict(name="cfg4_96c4", L=96, T=4, channels="all52", flavours=dict(u=(5, 0, 0.2), d="u", s=(5, 1, 0.3))),
]


def config_slice(cfg: dict, t: int, L: int | None = None) -> dict:
    """Draw u, d, s for time slice t of a CONFIGS entry.  Aliased flavours return the SAME array
    object (u=d means one draw, not two).  `L` overrides the lattice size (reduced-size tests)."""
    L = cfg["L"] if L is None else L
    out: dict[str, np.ndarray] = {}
    for f in "uds":
        spec = cfg["flavours"][f]
        if isinstance(spec, str):
            out[f] = out[spec]
        else:
            seed, stream, mass = spec
            out[f] = propagator(seed, stream, t, L, mass)
    return out
