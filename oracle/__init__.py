"""float64 CPU oracle -- TEST INFRASTRUCTURE ONLY (see crown_oracle.py header)."""
