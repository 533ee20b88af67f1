"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see mdwf_oracle.py / mdwf_oracle.c headers)."""
