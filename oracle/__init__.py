"""fp64 CPU oracle of the flag-and-average path (test infrastructure, not the product)."""
