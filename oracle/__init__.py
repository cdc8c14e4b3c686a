"""CPU oracle of the pseudo-spectral SPDE step — TEST INFRASTRUCTURE ONLY (see opss.h)."""
