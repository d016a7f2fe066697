// kernel instantiations: family c3 (configs[2]), N = 1..6 specialised + runtime N
#include "zmc_kernel.cuh"
namespace zmc {
extern const KernelEntry kEntriesC3[] = {
    ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 1, FamC3), ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 2, FamC3),
    ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 3, FamC3), ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 4, FamC3),
    ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 5, FamC3), ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 6, FamC3),
    ZMC_ENTRY_NDIM(ZMC_FAM_C3_OSCILLATORY, 0, FamC3),
};
extern const int kNumEntriesC3 = sizeof(kEntriesC3) / sizeof(kEntriesC3[0]);
}
