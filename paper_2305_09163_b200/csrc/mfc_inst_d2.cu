// kernels of the 2D template set
#define MFC_D 2
#include "mfc_inst.cuh"
