"""fp64 CPU oracle for the nodal-DG hot path of arxiv 1602.07997.

TEST INFRASTRUCTURE ONLY.  This package is the plain, slow, obviously-correct
restatement of what the hot path computes (volume term + upwind surface term
+ LSRK(5,4) update for the 3-D acoustic and isotropic elastic systems on
tetrahedra), written from the paper in numpy/fp64.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import it.  The product path
(``paper_1602_07997_b200``) never imports, links or executes anything here,
and nothing here imports the product path or the input generators.

Modules
-------
refelem  : reference tetrahedron: warp-and-blend nodes, orthonormal Dubiner
           basis, D_r/D_s/D_t, mass, face masks, merged LIFT  (PAPER.md:88-106,
           eq. (1)-(3); definitions the paper defers to its ref [33] follow
           DESIGN.md readings Q3/Q4)
mesh     : geometric factors g^vol, g^sur, normals, node coordinates,
           face-node connectivity by physical position
physics  : acoustic and elastic right-hand sides r_k (PAPER.md:36-84,
           eq. (5)-(6) and the two unnumbered elastic equations at 156-158)
timestep : LSRK(5,4) Carpenter-Kennedy update, stable dt, discrete energy
           (BASELINE.json north_star; readings Q1/Q2/Q10)

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): exact differentiation of
monomials, SPD mass matrix and quadrature orthonormality, summation-by-parts,
M*LIFT=E, interface Riemann solves, semi-discrete energy decay, standing-mode
convergence order, LSRK order conditions.  No function here is "parity
unpinned"; see DESIGN.md section "Oracle pins" for the map function -> pin.
"""
