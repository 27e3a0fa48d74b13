"""TEST INFRASTRUCTURE: float64 CPU oracle of the TACAW hot path (see tacaw_oracle.py).
Never imported by the product path (`paper_2602_10064_b200/`)."""
