"""Writes tests/golden/ising_dos_L{4,8,16,32}.txt: exact g(E_j), one integer per line, j = 0..N.

Source of the values: the closed form in tests/exact_dos.py (Kaufman/Beale, the
paper's own ground truth: PAPER.md:129, :215-221, ref. [43] at :305), evaluated
with mpmath and self-checked (sum = 2^N, symmetry, g0..g3).  Nothing here calls
the CUDA path or the oracle.  Run:  python tests/golden/make_dos_golden.py
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
import exact_dos  # noqa: E402

for L in (4, 8, 16, 32):
    g = exact_dos.exact_g(L)
    path = os.path.join(HERE, f"ising_dos_L{L}.txt")
    with open(path, "w") as f:
        f.write(f"# exact number of states g(E_j), E_j = -2N + 4j, j = 0..N, L = {L} periodic square-lattice Ising\n")
        f.write("# closed form: Kaufman/Beale (PAPER.md:129, :305 ref [43]); written by tests/golden/make_dos_golden.py\n")
        for v in g:
            f.write(f"{v}\n")
    print(path, len(g))
