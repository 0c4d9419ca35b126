"""CPU oracle for the DFT++ H.psi hot path -- TEST INFRASTRUCTURE ONLY (see jdft_ref.c / ref.py)."""
