"""CPU oracle for the demagnetizing-field convolution H_d = -N * M.

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_2008_02478_b200/`` imports,
links or executes this package, and this package imports nothing from there.
Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may call it.

What it computes (Table 1, "Demagnetizing Field"):

    H(r0) = - sum_r N(r - r0) M(r)

with N "computed using formulas in Ref. [50]" (Newell, Williams
and Dunlop 1993 — the formulas themselves are not printed in the paper, they
are restated in ``oracle/newell.py``), evaluated

* as the plain double sum (``oracle/demag_direct.py``) — the definition, and
* through the convolution theorem exactly as PAPER.md:L275 words it ("a (2)3D
  fast Fourier transform ... multiplied with the demagnetizing kernel in the
  transform space ... inverse (2)3D FFT"), with the zero padding of
  PAPER.md:L283, using an unpruned library FFT in fp64
  (``oracle/demag_fft.py``).  It is an accelerator for large meshes and is
  itself checked against the double sum.

``oracle/demag_pbc.py`` adds periodic boundary conditions by the multiple-images
method (Ref. [51]): the same sum over a finite block of copies of the
mesh, pinned in ``tests/test_oracle_pbc.py`` (the non-periodic double sum over the
tiled macro-geometry, trace, the infinite-film limit).

``oracle/multilayer.py`` is the multi-layered convolution of PAPER.md:L71-L76 (Eq. 4)
for a stack of one-cell-thick layers of unequal thickness at arbitrary heights
(reading R17), pinned in ``tests/test_oracle_multilayer.py`` (brute-force
quadrature between unequal cuboids, additivity, reciprocity, the single-mesh double
sum on a stack that sits on a common grid).

All arithmetic is fp64; the tensor is evaluated in x87 extended precision
(numpy.longdouble) because the closed form cancels catastrophically with
distance (reading R3).

Parity pins: every function here is pinned by ``tests/test_oracle_*.py``
against something other than itself (Aharoni's closed form for the prism
self-demagnetizing factor, brute-force 6-D quadrature of the dipolar kernel,
the point-dipole limit, trace/parity/permutation identities, the uniform-body
identity, the direct sum vs the FFT route, energy closed form).  Nothing here
is "parity unpinned".
"""
