"""Physical constants (cgs, CODATA 2018 exact SI values converted) used by the input recipes."""


class CGS:
    c = 2.99792458e10          # cm / s
    h = 6.62607015e-27         # erg s
    k_B = 1.380649e-16         # erg / K
    eV = 1.602176634e-12       # erg
    kpc = 3.0856775814913673e21  # cm
    Mpc = 3.0856775814913673e24  # cm
    yr = 3.15576e7             # s (Julian year)
    Myr = 3.15576e13
    E_HI_eV = 13.6             # hydrogen threshold used by the paper ("E_13.6")
