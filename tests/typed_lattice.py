"""Velocity sets and weights typed by hand, for the brute-force pins.

The brute-force gathers in tests/test_oracle_*_pins.py must not take their lattice from `oracle.lattice()`: that table
is part of what they pin.  D2Q9 is Eq. 3-4 as printed; D3Q19 / D3Q27 follow DESIGN.md R4 (lexicographic over
(e_x, e_y, e_z), each -1, 0, +1, e_x outermost; D3Q19 without the 8 corners); weights by |e|^2 (P:43, P:49 refs).
"""
import itertools

import numpy as np

E9 = [(-1, -1, 0), (-1, 0, 0), (-1, 1, 0), (0, -1, 0), (0, 0, 0), (0, 1, 0), (1, -1, 0), (1, 0, 0), (1, 1, 0)]
E19 = [(-1, -1, 0), (-1, 0, -1), (-1, 0, 0), (-1, 0, 1), (-1, 1, 0),
       (0, -1, -1), (0, -1, 0), (0, -1, 1), (0, 0, -1), (0, 0, 0), (0, 0, 1), (0, 1, -1), (0, 1, 0), (0, 1, 1),
       (1, -1, 0), (1, 0, -1), (1, 0, 0), (1, 0, 1), (1, 1, 0)]
E27 = list(itertools.product((-1, 0, 1), repeat=3))
WEIGHT_BY_SPEED2 = {9: (4 / 9, 1 / 9, 1 / 36), 19: (1 / 3, 1 / 18, 1 / 36), 27: (8 / 27, 2 / 27, 1 / 54, 1 / 216)}


def typed_lattice(Q):
    """(E, T): E a list of Q integer triples, T a float64 array of the Q weights."""
    E = {9: E9, 19: E19, 27: E27}[Q]
    T = np.array([WEIGHT_BY_SPEED2[Q][sum(abs(c) for c in v)] for v in E], dtype=np.float64)
    return E, T
