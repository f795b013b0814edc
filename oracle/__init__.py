"""CPU oracle for the hot path (test infrastructure, not the product).  See hot_oracle.c."""
