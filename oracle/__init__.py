"""The CPU oracle (test infrastructure only; see oracle/axo_oracle.cpp).  Not imported by the product path."""
