"""Physical constants and the model-table loader of the oracle.

Constants: SURVEY.md 8(c) "Constants [R]" (IAU/CODATA values; PAPER.md:47 arm
length 2.5 Gm; PAPER.md:81 10 yr = 3.15576e8 s fixes the Julian year).
"""
import os

C_SI = 299792458.0                    # m/s
MTSUN_S = 4.925491025543576e-06       # G Msun / c^3 in seconds
PC_M = 3.0856775814913674e16          # parsec in metres
GPC_S = 1.0e9 * PC_M / C_SI           # one Gpc in light-seconds
AU_M = 149597870700.0                 # astronomical unit in metres
AU_S = AU_M / C_SI                    # ... in light-seconds
ARM_M = 2.5e9                         # LISA arm length
ARM_S = ARM_M / C_SI                  # L/c
YEAR_SIDEREAL_S = 31558149.7635       # orbital period of the constellation
YEAR_JULIAN_S = 31557600.0            # "yr" of T_obs
EULER_GAMMA = 0.5772156649015328606

MODES = ((2, 2), (3, 3), (4, 4), (2, 1), (3, 2), (4, 3))   # PAPER.md:122, this order

_TABLE_PATH = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))),
                           "model_data", "phenomhm_table.csv")


def load_model_table(path=_TABLE_PATH):
    """Returns {name: float} from the CSV data file (name,value,provenance)."""
    table = {}
    with open(path) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, value, _tag = line.split(",")
            table[name] = float(value)
    return table
