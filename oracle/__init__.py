"""CPU oracle of the CooLBM lattice Boltzmann update.  TEST INFRASTRUCTURE, NOT THE PRODUCT."""
