"""ORACLE package: plain CPU implementation of the scheme (test infrastructure, not the product)."""
