// kernel instantiations: families c4, c5 (configs[3], configs[4])
#include "zmc_kernel.cuh"
namespace zmc {
extern const KernelEntry kEntriesC45[] = {
    ZMC_ENTRY_FIXED(ZMC_FAM_C4_GAUSS_PEAK, 6, FamC4),
    ZMC_ENTRY_FIXED(ZMC_FAM_C5_DAMPED_COS, 3, FamC5),
};
extern const int kNumEntriesC45 = sizeof(kEntriesC45) / sizeof(kEntriesC45[0]);
}
