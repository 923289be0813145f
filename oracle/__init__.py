"""CPU oracle for the KVarN hot path -- test infrastructure only (see kvarn_oracle.py)."""
