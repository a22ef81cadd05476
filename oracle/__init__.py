"""CPU oracle for the Walsh-Fourier PGD hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2606_06656_b200`` and neither imports the other.

* ``afs_oracle.c``     plain C, fp64: eq. (3) coefficients, literal (ESP) and count-basis evaluators,
                       objective/gradient, PGD, rounding and satisfaction counts (OpenMP over restarts).
* ``coeffs_exact.py``  exact rationals: brute-force Walsh transform, eq. (3), Appendix A closed forms.
* ``ref.py``           ctypes wrapper around the C file (numpy in, numpy out).
* ``build.py``         ``gcc -O2 -fopenmp -shared`` of the C file.
"""
