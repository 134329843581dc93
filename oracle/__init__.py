"""ORACLE: CPU reference of the FP8 EAGLE verify step.  Test infrastructure only - see
oracle/verify_oracle.py.  Nothing under paper_2606_18502_b200/ may import this package."""
