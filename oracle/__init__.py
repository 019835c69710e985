"""SharQ CPU oracle (test infrastructure only; see sharq_oracle.py header)."""
