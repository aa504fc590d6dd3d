"""CPU oracle for the convective-RHS hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  The product (``paper_2403_05910_b200``) never does, and this package never imports it.
The arithmetic lives in ``xf_oracle.c`` (plain C, fp64, ``-O2 -ffp-contract=off``); this file only builds it
with gcc, loads it with ctypes and marshals numpy arrays.
"""
from .oracle import Oracle, build, lib, OPrim, OConfig, OTransport, make_transport, OMechanism, make_mechanism, weno5, wenocu6, weno7  # noqa: F401
