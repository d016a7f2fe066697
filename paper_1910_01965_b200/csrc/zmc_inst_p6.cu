// kernel instantiations: the paper's family sin(sum y + sum x) (PAPER.md:75 Eq. 2, :120 Eq. 4)
#include "zmc_kernel.cuh"
namespace zmc {
extern const KernelEntry kEntriesP6[] = {
    ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 1, FamP6), ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 2, FamP6),
    ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 3, FamP6), ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 4, FamP6),
    ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 5, FamP6), ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 6, FamP6),
    ZMC_ENTRY_NDIM(ZMC_FAM_P6_SIN_SUM, 0, FamP6),
};
extern const int kNumEntriesP6 = sizeof(kEntriesP6) / sizeof(kEntriesP6[0]);
}
