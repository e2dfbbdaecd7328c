"""CPU oracle (test infrastructure, not the product).  See oracle.cpp header."""
