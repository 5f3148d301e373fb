"""CPU oracle of the Triad-ATRG hot path -- TEST INFRASTRUCTURE ONLY (see tatrg_oracle.py)."""
