"""fp64 CPU oracle for the batched-LM hot path.  TEST INFRASTRUCTURE ONLY -- see lm_oracle.h."""
