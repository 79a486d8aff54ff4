"""Writes the small text fixtures in this folder.  Each value is a closed form
the paper prints (no oracle, no CUDA involved): run `python tests/golden/make_golden.py`."""
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))

with open(os.path.join(HERE, "eq12_inclined_disk.txt"), "w") as f:
    f.write("# PAPER.md:135 eq. 12 (sec. 3.1): p = sin^2 i / (2 + sin^2 i); columns: i [deg], p\n")
    for i in (0, 10, 20, 30, 45, 60, 70, 80, 90):
        s = math.sin(math.radians(i)) ** 2
        f.write("%d %.7f\n" % (i, s / (2 + s)))
