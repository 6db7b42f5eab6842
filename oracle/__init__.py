"""CPU oracle (test infrastructure only; see pvf_oracle.py header).  Never imported by the product."""
