"""CPU ORACLE for the FEnc^2 CKKS hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2606_16359_b200/ and never
imports it.  See DESIGN.md section 4 for the readings (R2.x / A-n) cited in docstrings.
"""
