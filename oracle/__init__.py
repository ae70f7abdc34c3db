"""CPU fp64 oracle for the MUSER dirty-imaging hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
See muser_oracle.py (numpy transcription, whole path) and oracle_c.c (+ oracle_c.py ctypes wrapper;
plain-C transcription of the gridder and the direct DFT for full-size configs and timing)."""
