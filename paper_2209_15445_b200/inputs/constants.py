"""Physical constants and the log-energy grid (SURVEY.md §8 header; BASELINE.json:north_star).

Units: energy MeV, length cm, field tesla, density g/cm^3.
This module belongs to the *input builder*: it produces the inputs (tables, geometry,
field, primaries) that both the CUDA library and the test oracle consume.  It holds
none of the per-step transport arithmetic.
"""
import math

ELECTRON_MASS = 0.51099895            # m_e c^2 [MeV]
R_E = 2.8179403262e-13                # classical electron radius [cm]
ALPHA = 1.0 / 137.035999084           # fine-structure constant
N_AVOGADRO = 6.02214076e23            # [1/mol]
C_B = 2.99792458                      # p[MeV/c] = C_B * B[T] * R[cm]
RYDBERG_EV = 13.605693                # [eV]

# 2048-point grid uniform in u = ln T from 1 keV to 100 TeV (north_star)
N_GRID = 2048
T_GRID_MIN = 1.0e-3
T_GRID_MAX = 1.0e8
U0 = math.log(T_GRID_MIN)
DU = (math.log(T_GRID_MAX) - math.log(T_GRID_MIN)) / (N_GRID - 1)

PRODUCTION_CUT_CM = 0.07              # 0.7 mm (north_star)

# table order inside one material block: 12 x double[2048]
TAB_G_COMPTON, TAB_G_PAIR, TAB_G_PHOTO = 0, 1, 2
TAB_EM_BREM, TAB_EM_IONI, TAB_EM_DEDX, TAB_EM_RANGE = 3, 4, 5, 6
TAB_EP_BREM, TAB_EP_IONI, TAB_EP_ANNI, TAB_EP_DEDX, TAB_EP_RANGE = 7, 8, 9, 10, 11
N_TABLES = 12

# species codes of the C ABI
ELECTRON, POSITRON, GAMMA = 0, 1, 2
