"""CPU oracle for the Chebyshev-filtered spinor H.X (test infrastructure, not the product)."""
