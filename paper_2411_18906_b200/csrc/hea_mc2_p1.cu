// hea_mc2_p1.cu -- part 1 of the halo-engine instantiations (lattice bcc, lowest-index selection); see hea_mc2.cu.
#define HEA_MC2_PART 1
#include "hea_mc2.cu"
