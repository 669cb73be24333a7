"""CPU oracle of the gateau hot path -- TEST INFRASTRUCTURE ONLY (see oracle/gateau_oracle.h)."""
