"""CPU oracle for the phase-space source hot path -- TEST INFRASTRUCTURE ONLY.

See psl_oracle.c for the definition and its citations.  Nothing under paper_1302_1861_b200/
imports this package, and this package imports nothing from it.
"""
