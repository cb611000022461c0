"""Seeded primary generators for the five synthetic workloads.

Every random attribute of event i comes from the generator stream (event i, track id 2^64-1,
step 0), consumed sequentially per primary in the order (species, energy, phi, eta, y0, z0) as far
as the config uses them.  Output: dict of numpy arrays (event, species, pos, dir, ekin).
"""
import math

import numpy as np

from .constants import ELECTRON, GAMMA, POSITRON
from .philox import uniforms

GEN_TRACK = (1 << 64) - 1


def _pack(event, species, pos, direc, ekin):
    return {"event": np.ascontiguousarray(event, dtype=np.uint32),
            "species": np.ascontiguousarray(species, dtype=np.int8),
            "pos": np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3),
            "dir": np.ascontiguousarray(direc, dtype=np.float64).reshape(-1, 3),
            "ekin": np.ascontiguousarray(ekin, dtype=np.float64)}


def beam(n_events, ekin, species=ELECTRON, spread=0.0, seed=1, first_event=0):
    """Configs 1-3: one primary per event along +x from the front face; y0,z0 = spread(-1+2U)."""
    pos = np.zeros((n_events, 3))
    if spread > 0.0:
        for e in range(n_events):
            u = uniforms(first_event + e, seed, GEN_TRACK, 0, 2)
            pos[e, 1] = spread * (-1.0 + 2.0 * u[0])
            pos[e, 2] = spread * (-1.0 + 2.0 * u[1])
    d = np.zeros((n_events, 3)); d[:, 0] = 1.0
    return _pack(first_event + np.arange(n_events), np.full(n_events, species), pos, d,
                 np.full(n_events, float(ekin)))


def _eta_phi_dir(eta, phi):
    theta = 2.0 * np.arctan(np.exp(-eta))
    return np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)], axis=-1)


def barrel_events(n_events, n_per_event, e_lo, e_hi, mode="cfg4", seed=1, first_event=0, eta_max=1.4):
    """Configs 4-5: primaries from the origin, ln T uniform, phi uniform, eta uniform in (-1.4,1.4).

    mode "cfg4": species e-/gamma by U < 1/2 (4 draws per primary: species, energy, phi, eta);
    mode "cfg5": species by (index mod 5): 0,1 -> e-, 2 -> e+, 3,4 -> gamma (3 draws per primary).
    """
    ev, sp, ek, dr = [], [], [], []
    per = 4 if mode == "cfg4" else 3
    for e in range(n_events):
        u = uniforms(first_event + e, seed, GEN_TRACK, 0, per * n_per_event).reshape(n_per_event, per)
        if mode == "cfg4":
            species = np.where(u[:, 0] < 0.5, ELECTRON, GAMMA)
            ue, up, uh = u[:, 1], u[:, 2], u[:, 3]
        else:
            species = np.array([ELECTRON, ELECTRON, POSITRON, GAMMA, GAMMA])[np.arange(n_per_event) % 5]
            ue, up, uh = u[:, 0], u[:, 1], u[:, 2]
        ekin = np.exp(math.log(e_lo) + ue * (math.log(e_hi) - math.log(e_lo)))
        phi = 2.0 * math.pi * up
        eta = -eta_max + 2.0 * eta_max * uh
        ev.append(np.full(n_per_event, first_event + e)); sp.append(species); ek.append(ekin)
        dr.append(_eta_phi_dir(eta, phi))
    n = n_events * n_per_event
    return _pack(np.concatenate(ev), np.concatenate(sp), np.zeros((n, 3)), np.concatenate(dr),
                 np.concatenate(ek))
