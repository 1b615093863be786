"""CPU oracle for the MEB hot path  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct numpy implementation (float64 unless a function says
otherwise) of what the CUDA path computes, written from /root/reference/PAPER.md
("Mixed-Precision GPU Acceleration for Large-Scale Minimum Enclosing Ball Problems").
Citations ``P:L<n>`` are PAPER.md line numbers.

Rules (see the task statement, section (3)):

* Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
  ``--impl reference`` legs may import this package.  The product path
  (``paper_2605_31425_b200``) never does, and fails loudly without its CUDA library.
* It shares no code with the CUDA path.  Only ``workloads`` (seeded input generators,
  no method arithmetic) serves both.
* There is no blocking, fusion or reordering beyond what the formulas state.

Modules
-------
``soc``         second-order-cone projection, distance, Clarke Jacobian element.
``primitives``  eval_alm, hvp, dense_hessian, update_multipliers, screen, compact,
                feasibility_check: one plain pass over the balls each.
``ripalm``      Algorithm 1, Algorithm 2, the mixed-precision
                reduction loop and ``meb_solve``.

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): closed forms, brute force in d=2,
finite differences, Moreau decomposition, weak-duality certificate, Table 1 of the paper.
Parity unpinned (items 3-5 and 10-12): the solver's free constants
(rho, sigma_0, kappa, tau, Armijo constants, CG tolerance, caps).  They change the
iteration path, not the answer; the answer is pinned.  The CUDA path additionally has two
safeguards the oracle does not need at test sizes (DESIGN readings 17 and 18: a capped
low-precision run, best-iterate / stall logic); they too change the path only.
"""
