"""CPU oracle for the MSD-AFQMC hot path (arXiv 2406.08314).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_2406_08314_b200/`` imports,
links or executes anything in this directory; only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may.  It shares no code with the CUDA path: the only common
module is ``msd_inputs`` (seeded input generators, no method arithmetic).

Tiers (all follow PAPER.md Eq. 2, 7, 13-15 and L98/L114:
"performing SD-AFQMC for each individual determinant"):

  O0  oracle.msd_oracle.o0_pure_determinants   explicit determinants only
  O1  oracle.msd_oracle.o1_definition          dense N x N Green's function per determinant
  O2  oracle.o2 (C, OpenMP; liboracle_o2.so)   same maths touching only non-zero rows

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): Fock-space brute force of
Eq. 2/7/13-15 on micro inputs, Eq. 2 == Eq. 3+4, single-determinant closed
forms, gauge invariance, Hartree-Fock limit, O0 == O1 == O2.  The paper prints
no worked numerical example, so beyond those pins parity is unpinned against
the authors' own numbers.
"""
