// chisao_eval_obj.cu -- instantiates the evaluation kernels for ONE objective id
// (compiled six times with -DCHISAO_OBJ_INST=0..5; 5 = the Appendix-D family so the translation units build in parallel).
#include "chisao_eval_kernels.cuh"
#include "chisao_resident.cuh"

#ifndef CHISAO_OBJ_INST
#error "compile with -DCHISAO_OBJ_INST=<objective id>"
#endif

#define CHISAO_CAT2(a, b) a##b
#define CHISAO_CAT(a, b) CHISAO_CAT2(a, b)

namespace chisao {

cudaError_t CHISAO_CAT(launch_fd_obj_, CHISAO_OBJ_INST)(const DevObj &o, const FdArgs &a, int grid, cudaStream_t st) {
  return launch_fd_obj<CHISAO_OBJ_INST>(o, a, grid, st);
}
cudaError_t CHISAO_CAT(launch_pt_obj_, CHISAO_OBJ_INST)(const DevObj &o, const PtArgs &a, int grid, cudaStream_t st) {
  return launch_pt_obj<CHISAO_OBJ_INST>(o, a, grid, st);
}
cudaError_t CHISAO_CAT(launch_hlc_obj_, CHISAO_OBJ_INST)(const DevObj &o, const HlcArgs &a, int grid, cudaStream_t st) {
  return launch_hlc_obj<CHISAO_OBJ_INST>(o, a, grid, st);
}
cudaError_t CHISAO_CAT(configure_obj_, CHISAO_OBJ_INST)() { return configure_obj<CHISAO_OBJ_INST>(); }
cudaError_t CHISAO_CAT(launch_resident_obj_, CHISAO_OBJ_INST)(const DevObj &o, const ResArgs &a, cudaStream_t st) {
  return launch_resident_obj<CHISAO_OBJ_INST>(o, a, st);
}
cudaError_t CHISAO_CAT(configure_resident_obj_, CHISAO_OBJ_INST)() { return configure_resident_obj<CHISAO_OBJ_INST>(); }

}  // namespace chisao
