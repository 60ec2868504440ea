// Instantiations of the register-resident solve kernel (pca_reg.cuh), split over several translation
// units (-DPCA_REG_PART=0..5) so that they compile in parallel.  NV = 2 (eight columns per thread and row).
#include "pca_one.cuh"

#ifndef PCA_REG_PART
#error "compile with -DPCA_REG_PART=<0..5>"
#endif

namespace pca {

#define PCA_RV(GT, RPT) \
  if (gt == GT && rpt == RPT) return pca_reg_kernel<GT, 2, RPT>;
#define PCA_RV3(GT) PCA_RV(GT, 2) PCA_RV(GT, 4) PCA_RV(GT, 7)

#define PCA_OV(GT, RPT) \
  if (gt == GT && rpt == RPT) return pca_one_kernel<GT, RPT>;
#define PCA_OV3(GT) PCA_OV(GT, 2) PCA_OV(GT, 4) PCA_OV(GT, 7)

#define PCA_RVS(GT) \
  if (gt == GT) return pca_reg_kernel<GT, 2, 7, kRegSmemRows>;

#if PCA_REG_PART == 0
reg_kernel_t reg_kernel_lookup_part0(int gt, int rpt) {
  PCA_RV3(8) PCA_RV3(16)
  return nullptr;
}
one_kernel_t one_kernel_lookup_part0(int gt, int rpt) {
  PCA_OV3(8) PCA_OV3(16)
  return nullptr;
}
#elif PCA_REG_PART == 1
reg_kernel_t reg_kernel_lookup_part1(int gt, int rpt) {
  PCA_RV3(32) PCA_RV3(64)
  return nullptr;
}
one_kernel_t one_kernel_lookup_part1(int gt, int rpt) {
  PCA_OV3(32) PCA_OV3(64)
  return nullptr;
}
#elif PCA_REG_PART == 2
reg_kernel_t reg_kernel_lookup_part2(int gt, int rpt) {
  PCA_RV3(128) PCA_RV(256, 7)
  return nullptr;
}
#elif PCA_REG_PART == 3
reg_kernel_t reg_kernel_lookup_part3(int gt, int rpt) {
  PCA_RV(256, 2) PCA_RV(256, 4) PCA_RV3(512)
  return nullptr;
}
// the RPT = 7 variants with kRegSmemRows rows of the row block in shared memory (fewer spills; the plan takes them when shared
// memory is not needed for the panels)
#elif PCA_REG_PART == 4
reg_kernel_t reg_kernel_lookup_part4(int gt) {
  PCA_RVS(8) PCA_RVS(16) PCA_RVS(32) PCA_RVS(64)
  return nullptr;
}
#else
reg_kernel_t reg_kernel_lookup_part5(int gt) {
  PCA_RVS(128) PCA_RVS(256) PCA_RVS(512)
  return nullptr;
}
#endif

}  // namespace pca
