"""Writes tests/golden/inflow_hash_pins.txt: eight values of the oracle's counter-based inflow-noise generator
(reading O1), as exact hex floats.  Calls only oracle/.

    python tests/golden/make_inflow_hash_pins.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import oracle as O  # noqa: E402

CASES = [(2024, 0, 0, 0, 0), (2024, 1, 0, 0, 0), (2024, 0, 0, 1, 0), (2024, 0, 0, 0, 1), (2024, 49, 0, 255, 31),
         (3, 5, 2, 17, 4), (12345, 1000000, 1, 127, 127), (0, 0, 5, 2, 9)]

with open(os.path.join(HERE, "inflow_hash_pins.txt"), "w") as f:
    f.write("# seed step face a b value(hex float) -- oracle.inflow_rand, written by make_inflow_hash_pins.py\n")
    for c in CASES:
        f.write("%d %d %d %d %d %s\n" % (c + (float(O.inflow_rand(*c)).hex(),)))
