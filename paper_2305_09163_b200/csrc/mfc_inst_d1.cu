// kernels of the 1D template set
#define MFC_D 1
#include "mfc_inst.cuh"
