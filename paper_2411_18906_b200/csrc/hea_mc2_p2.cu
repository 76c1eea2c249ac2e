// hea_mc2_p2.cu -- part 2 of the halo-engine instantiations (lattice fcc, best-of-K selection); see hea_mc2.cu.
#define HEA_MC2_PART 2
#include "hea_mc2.cu"
