"""CPU fp64 oracle for the SFT inner product of arXiv:2502.11823 (Tenorio & Gerosa).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import it.  It shares no code, table or constant generator with the CUDA
path in ``paper_2502_11823_b200/`` and never imports it.

Everything is plain numpy in fp64 and follows the paper's equations in the paper's
order (citations ``P:NNN`` are line numbers of ``/root/reference/PAPER.md``):

* ``oracle.waveform``  – restricted TaylorT3 inspiral (0PN / 0PN+1PN): the four numbers
  ``{A, phi, f, fdot}`` per SFT of P:164, plus the SFT-length rule Eq.(34) P:248.
* ``oracle.kernel``    – the kernel ``Fre`` by its definition Eq.(28) P:215 (quadrature),
  its closed form Eq.(29)-(32) P:219-236, the discrete sum Eq.(27) P:208 and the
  Dirichlet limit Eq.(B2) P:451.
* ``oracle.sft``       – data SFTs by direct DFT, Eq.(26), and the plain
  time-domain / full-band inner products Eq.(1), Eq.(14) P:149.
* ``oracle.inner``     – the method itself, Eq.(20)/(24)/(35) P:178-259 with the band
  truncation of P:238, and the cumulative-over-SFTs variant.
* ``oracle.stats``     – log-likelihood Eq.(2), phase-maximised statistic Eq.(7)-(9), F-statistic Eq.(10)-(13) P:63-122
  (all 4 + 10 products bin by bin, plain 4 x 4 solve).
* ``oracle.accuracy``  – the accuracy experiment of section IV: ``<d,h>`` by direct integration and ``r`` of Eq.(36) P:274.
  (``oracle.sft`` also holds the per-SFT noise-level estimate of P:139, ``oracle.inner`` the validity measure of Eq.(33).)

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``) tie each function to something
other than itself; a function without such a pin says "parity unpinned" in its
docstring.
"""
