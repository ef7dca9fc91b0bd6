"""Physical constants and detector geometry used by the oracle (test infrastructure).

None of these numbers is printed in PAPER.md; they are the DESIGN.md "readings" R-C1 (constants)
and R-P3 (site geometry).  The detectors are the ones the paper names: Hanford, Livingston
 and Virgo ("LIGO-Virgo").
"""
import numpy as np

C_SI = 299792458.0                       # m/s (exact)
MTSUN_SI = 4.925490947641267e-06         # G*Msun/c^3 in seconds (IAU nominal GM_sun)
MRSUN_SI = MTSUN_SI * C_SI               # G*Msun/c^2 in metres
MPC_SI = 3.085677581491367e22            # metres per megaparsec
EULER_GAMMA = 0.5772156649015329

# Earth-fixed vertex position (m) and arm unit vectors; index 0 = H1, 1 = L1, 2 = V1.
DETECTORS = {
    0: dict(name="H1",
            r=np.array([-2.16141492636e6, -3.83469517889e6, 4.60035022664e6]),
            x=np.array([-0.22389266154, 0.79983062746, 0.55690487831]),
            y=np.array([-0.91397818574, 0.02609403989, -0.40492342125])),
    1: dict(name="L1",
            r=np.array([-7.42760447238e4, -5.49628371971e6, 3.22425701744e6]),
            x=np.array([-0.95457412153, -0.14158077340, -0.26218911324]),
            y=np.array([0.29774156894, -0.48791033647, -0.82054461286])),
    2: dict(name="V1",
            r=np.array([4.54637409900e6, 8.42989697626e5, 4.37857696241e6]),
            x=np.array([-0.70045821479, 0.20848948619, 0.68256166277]),
            y=np.array([-0.05379255368, -0.96908180549, 0.24080451708])),
}
