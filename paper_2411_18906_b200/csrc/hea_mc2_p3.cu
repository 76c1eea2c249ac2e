// hea_mc2_p3.cu -- part 3 of the halo-engine instantiations (lattice bcc, best-of-K selection); see hea_mc2.cu.
#define HEA_MC2_PART 3
#include "hea_mc2.cu"
