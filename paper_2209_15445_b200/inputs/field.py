"""Magnetic-field descriptors (BASELINE.json:configs[2],[3])."""
from dataclasses import dataclass, field as _f

import numpy as np

FIELD_NONE, FIELD_UNIFORM, FIELD_MAP_RZ = 0, 1, 2


@dataclass
class Field:
    kind: int = FIELD_NONE
    B: tuple = (0.0, 0.0, 0.0)                 # uniform field [T]
    nr: int = 0
    nz: int = 0
    r0: float = 0.0
    z0: float = 0.0
    dr: float = 1.0
    dz: float = 1.0
    bz: np.ndarray = _f(default_factory=lambda: np.zeros(0))   # float64 [nz, nr], B = (0,0,bz)


def no_field():
    return Field()


def uniform_field(bx, by, bz):
    return Field(kind=FIELD_UNIFORM, B=(float(bx), float(by), float(bz)))


def solenoid_map(b0=3.8, r_scale=300.0, r_max=300.0, z_half=300.0, step=1.0):
    """Bz(r) = b0 (1 - (r/r_scale)^2) on a 1 cm r-z grid, r = 0..300, z = -300..300 (config 4)."""
    nr = int(round(r_max / step)) + 1
    nz = int(round(2.0 * z_half / step)) + 1
    r = step * np.arange(nr)
    prof = b0 * (1.0 - (r / r_scale) ** 2)
    bz = np.ascontiguousarray(np.tile(prof.reshape(1, nr), (nz, 1)))
    return Field(kind=FIELD_MAP_RZ, nr=nr, nz=nz, r0=0.0, z0=-z_half, dr=step, dz=step, bz=bz)
