"""ORACLE (test infrastructure): physical constants (readings S1, S2)."""
import math

MU0 = 4e-7 * math.pi          # T m / A (S2)
GAMMA = 1.7595e11             # rad / (T s) (S1; per-material parameter, this is the default)
MU_B = 9.2740100783e-24       # J / T
Q_E = 1.602176634e-19         # C
HBAR = 1.054571817e-34        # J s

# effective-field term bits (same numbering as include/mmx.h)
T_EXCH, T_DMI, T_ANIS_U, T_ANIS_C, T_ZEEMAN, T_DEMAG, T_A12, T_A0, T_DMI_INTER, T_MEL, T_DMI_HOMO = (
    1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1024)
T_ALL = 2047
TERM_BITS = dict(exch=T_EXCH, dmi=T_DMI, anis_u=T_ANIS_U, anis_c=T_ANIS_C, zeeman=T_ZEEMAN,
                 demag=T_DEMAG, a12=T_A12, a0=T_A0, dmi_inter=T_DMI_INTER, mel=T_MEL, dmi_homo=T_DMI_HOMO)
