"""CPU oracle for the single-GPU direct Poisson solve of arxiv 1909.05423 (PittPack).

TEST INFRASTRUCTURE ONLY.  Nothing under ``oracle/`` is part of the product path.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import it.  It shares no code with the CUDA path under
``paper_1909_05423_b200/`` and never imports it; expected values never come from the
CUDA path.

Contents
--------
``poisson_oracle``  the definition written out: naive O(n^2) per-axis transform sums
                    (PAPER.md:115, 128, 165 -- eq. 6, 7, 9), textbook Thomas
                    (Algorithm 1), Sherman-Morrison for periodic z
                    (PAPER.md:216), the zero-mode fix.
``makhoul``         the paper's three-step pre / complex-FFT / post recipes for the real
                    transforms, step by step in the paper's
                    order, used only to pin the readings of the garbled passages.

Parity pins: every function is pinned in ``tests/test_oracle_*.py`` against something
other than itself (Table 2 eigenpairs, literal loops over eq. 6-10, dense LU / pinv of
the Kronecker-assembled operator for all 27 BC combinations, closed-form eigenmode
solutions, the 20 printed errors of Tables 3-7).  No function is "parity unpinned".
"""
