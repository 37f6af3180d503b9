// kernels of the 3D template set
#define MFC_D 3
#include "mfc_inst.cuh"
