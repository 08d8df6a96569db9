"""CPU oracle (test infrastructure only; see fe_oracle.py header).  Never imported by the product path."""
