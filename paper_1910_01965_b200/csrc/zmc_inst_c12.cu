// kernel instantiations: families c1, c2 (BASELINE.json configs[0], configs[1])
#include "zmc_kernel.cuh"
namespace zmc {
extern const KernelEntry kEntriesC12[] = {
    ZMC_ENTRY_FIXED(ZMC_FAM_C1_COS_XY, 1, FamC1),
    ZMC_ENTRY_FIXED(ZMC_FAM_C2_SIN_XY2, 2, FamC2),
};
extern const int kNumEntriesC12 = sizeof(kEntriesC12) / sizeof(kEntriesC12[0]);
}
