"""CPU oracle (test infrastructure, not the product). See exc_oracle.py."""
