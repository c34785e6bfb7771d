"""Mode indexing (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

PAPER.md:236, 256: modes (l, m, p), l = 1..lmax, m = -l..l, p in {0, 1};
L = 2*lmax*(lmax+2) coefficients per scatterer.  The flat order is not stated in the
paper; reading R1 (part of the ABI): idx = p*(L/2) + l*(l+1) - 1 + m.
"""


def n_modes(lmax):
    return 2 * lmax * (lmax + 2)


def mode_index(l, m, p, lmax):
    return p * (n_modes(lmax) // 2) + l * (l + 1) - 1 + m


def mode_list(lmax):
    """[(l, m, p)] in flat order."""
    out = []
    for p in (0, 1):
        for l in range(1, lmax + 1):
            for m in range(-l, l + 1):
                out.append((l, m, p))
    return out
