"""CPU FP64 oracle for the TA-SC-IVR hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package.  It shares no code with paper_1312_4698_b200 (the CUDA path) and
neither imports the other; both take their inputs from paper_1312_4698_b200.inputs, which
holds none of the method's arithmetic.

  oracle.sc_ivr_oracle.c   the step-by-step C implementation (one loop nest per formula)
  oracle.capi              ctypes access to it (builds liboracle in-tree with gcc on demand)
  oracle.brute             a second, independent, numpy-only single-trajectory implementation
                           built on library routines (numpy.linalg.det, numpy.unwrap, einsum
                           over the full coupling tensors) - the brute-force pin for tiny inputs
"""
