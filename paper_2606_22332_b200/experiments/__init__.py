"""Measured design experiments that are not on the product path (each is its own small shared library)."""
