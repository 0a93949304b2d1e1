"""Seeded synthetic inputs: flat RAMBO phase-space points and the parameter card.

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It holds none
of the method's arithmetic (no wavefunctions, no amplitudes, no colour algebra): it only
draws momenta, which both sides then read from the same buffer.

What it stands in for: the paper's `check.exe` draws random numbers and samples phase
space itself (Sec. 2.1) but never says how; BASELINE.json fixes the recipe
instead: flat RAMBO at sqrt(s) = 1500 GeV, seed 1, beams along +-z.

Algorithm (restated, not copied): R. Kleiss, W.J. Stirling, S.D. Ellis, "A new Monte
Carlo treatment of multiparticle phase space at high energies" (RAMBO): n isotropic
massless vectors with energies distributed as x*exp(-x), conformally boosted and scaled
to total momentum (sqrt(s), 0, 0, 0); masses are then introduced by rescaling all
three-momenta with one factor xi solving sum_i sqrt(m_i^2 + xi^2 |p_i|^2) = sqrt(s)
(Newton iteration).  The event weight is not needed here and is not computed.

Random numbers: numpy's Philox (a counter-based generator, key = seed), 4 uniform doubles
per final-state particle per event, drawn event-major, so that event i of a large batch
equals event i of a small one with the same seed.
"""
from __future__ import annotations

import numpy as np

# --- parameter card (BASELINE.json configs; PAPER.md never prints one) -----------------
PARAMS = {
    "aEWM1": 132.507,   # 1/alpha
    "mZ": 91.188,
    "wZ": 2.4414,
    "mW": 80.419,
    "mT": 173.0,
    "wT": 1.4915,
    "aS": 0.118,
}

SQRT_S = 1500.0

# name -> (final-state masses selector, number of final-state particles, nevt of the config)
# Particle order = order in the process string: two beams, then the final state.
PROCESSES = {
    #  name          final masses (keys into PARAMS or 0.0)        BASELINE.json nevt
    "epem_mupmum": {"final": [0.0, 0.0], "nevt": 16384},
    "gg_ttx": {"final": ["mT", "mT"], "nevt": 524288},
    "gg_ttxg": {"final": ["mT", "mT", 0.0], "nevt": 524288},
    "gg_ttxgg": {"final": ["mT", "mT", 0.0, 0.0], "nevt": 262144},
    "gg_ttxggg": {"final": ["mT", "mT", 0.0, 0.0, 0.0], "nevt": 65536},
    # SURVEY.md §8(f) row 3 (Table 2 and Tables 5-8 of the paper; not a BASELINE.json config): batch size chosen here
    "gg_ttxgggg": {"final": ["mT", "mT", 0.0, 0.0, 0.0, 0.0], "nevt": 4096},
}


def final_masses(process: str, params: dict | None = None) -> np.ndarray:
    p = dict(PARAMS)
    if params:
        p.update(params)
    return np.array([p[m] if isinstance(m, str) else float(m) for m in PROCESSES[process]["final"]],
                    dtype=np.float64)


def npar(process: str) -> int:
    return 2 + len(PROCESSES[process]["final"])


def _uniforms(seed: int, nevt: int, nfinal: int, first_event: int = 0) -> np.ndarray:
    """[nevt][nfinal][4] uniforms in (0,1); event i always gets the same numbers for a given seed."""
    bg = np.random.Philox(key=int(seed))
    # Philox yields 4 x 64-bit words per counter step and one double consumes one word, so
    # advancing by one step skips exactly 4 doubles = one final-state particle.
    bg.advance(int(first_event) * nfinal)
    gen = np.random.Generator(bg)
    u = gen.random((nevt, nfinal, 4))
    # keep strictly inside (0,1): log(0) must never occur
    np.clip(u, 2.0 ** -53, 1.0 - 2.0 ** -53, out=u)
    return u


def rambo(nevt: int, masses, sqrt_s: float = SQRT_S, seed: int = 1, first_event: int = 0) -> np.ndarray:
    """Flat RAMBO: returns momenta[nevt][2 + nfinal][4] as (E, px, py, pz) in GeV, fp64.

    Beams: p0 = (sqrt_s/2, 0, 0, +sqrt_s/2), p1 = (sqrt_s/2, 0, 0, -sqrt_s/2), massless.
    """
    masses = np.asarray(masses, dtype=np.float64)
    nf = masses.shape[0]
    u = _uniforms(seed, nevt, nf, first_event)
    c = 2.0 * u[..., 0] - 1.0
    s = np.sqrt(1.0 - c * c)
    f = 2.0 * np.pi * u[..., 1]
    e = -np.log(u[..., 2] * u[..., 3])
    q = np.empty((nevt, nf, 4))
    q[..., 0] = e
    q[..., 1] = e * s * np.cos(f)
    q[..., 2] = e * s * np.sin(f)
    q[..., 3] = e * c
    # conformal transformation to the centre-of-mass frame with invariant mass sqrt_s
    Q = q.sum(axis=1)                                     # [nevt][4]
    M = np.sqrt(Q[:, 0] ** 2 - Q[:, 1] ** 2 - Q[:, 2] ** 2 - Q[:, 3] ** 2)
    b = -Q[:, 1:] / M[:, None]                            # [nevt][3]
    x = sqrt_s / M
    gam = Q[:, 0] / M
    a = 1.0 / (1.0 + gam)
    bq = np.einsum("ej,enj->en", b, q[..., 1:])          # b . q_i
    p = np.empty_like(q)
    p[..., 0] = x[:, None] * (gam[:, None] * q[..., 0] + bq)
    p[..., 1:] = x[:, None, None] * (q[..., 1:] + b[:, None, :] * q[..., 0:1]
                                     + (a[:, None] * bq)[..., None] * b[:, None, :])
    # Remove the rounding left by the (ill-conditioned for near-collinear q_i) conformal boost:
    # re-centre the three-momenta so that they sum to zero exactly, then solve for the one scale
    # factor xi with sum_i sqrt(m_i^2 + xi^2 |p_i|^2) = sqrt_s (Newton).  For massless final
    # states xi = 1 up to that rounding; for massive ones this is RAMBO's mass rescaling.
    p[..., 1:] -= p[..., 1:].mean(axis=1, keepdims=True)
    m2 = masses ** 2
    e2 = (p[..., 1:] ** 2).sum(axis=-1)
    xi = np.full(nevt, np.sqrt(max(1.0 - (masses.sum() / sqrt_s) ** 2, 0.0)))
    for _ in range(16):          # fixed count (quadratic convergence): event i never depends on the batch
        en = np.sqrt(m2[None, :] + (xi ** 2)[:, None] * e2)
        f0 = en.sum(axis=1) - sqrt_s
        g0 = (xi[:, None] * e2 / en).sum(axis=1)
        xi -= f0 / g0
    p[..., 1:] *= xi[:, None, None]
    # put every final-state particle exactly on its mass shell: E = sqrt(m^2 + |p|^2)
    p[..., 0] = np.sqrt(masses[None, :] ** 2 + (p[..., 1:] ** 2).sum(axis=-1))
    out = np.empty((nevt, nf + 2, 4))
    out[:, 0] = (0.5 * sqrt_s, 0.0, 0.0, 0.5 * sqrt_s)
    out[:, 1] = (0.5 * sqrt_s, 0.0, 0.0, -0.5 * sqrt_s)
    out[:, 2:] = p
    return np.ascontiguousarray(out)


def momenta(process: str, nevt: int | None = None, seed: int = 1, first_event: int = 0,
            params: dict | None = None) -> np.ndarray:
    """Momenta for one of the five BASELINE.json configs (nevt defaults to the config's size)."""
    if nevt is None:
        nevt = PROCESSES[process]["nevt"]
    return rambo(nevt, final_masses(process, params), SQRT_S, seed, first_event)
