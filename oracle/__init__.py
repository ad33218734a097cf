"""CPU oracle for the HHS-FSI hot path -- TEST INFRASTRUCTURE ONLY (see frost_oracle.c header).

Thin ctypes marshalling over oracle/libfrost_oracle.so.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package; the product package
paper_2011_14984_b200 never does, and this package never imports it.
"""
from .frost_oracle import *  # noqa: F401,F403
