"""CPU oracle for the DD-4DVar hot path.  TEST INFRASTRUCTURE -- not imported by the product."""
from .oracle import Oracle, lbfgs_minimize  # noqa: F401
