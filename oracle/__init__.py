"""CPU oracle of the SWE finite-volume step.  TEST INFRASTRUCTURE, not the product."""
