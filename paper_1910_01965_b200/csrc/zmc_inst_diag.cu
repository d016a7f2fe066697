// kernel instantiations: diagnostic families (tests only), runtime N
#include "zmc_kernel.cuh"
namespace zmc {
extern const KernelEntry kEntriesDiag[] = {
    ZMC_ENTRY_DIAG(ZMC_FAM_CONST_ONE, FamConstOne), ZMC_ENTRY_DIAG(ZMC_FAM_PARAM_ECHO, FamParamEcho),
    ZMC_ENTRY_DIAG(ZMC_FAM_LIN_Y, FamLinY),         ZMC_ENTRY_DIAG(ZMC_FAM_POLY, FamPoly),
};
extern const int kNumEntriesDiag = sizeof(kEntriesDiag) / sizeof(kEntriesDiag[0]);
}
