// One translation unit per supported pencil length: compiled once for every MVD_LEN(A, B) line of
// lengths.def with -DMVD_INST_A=A -DMVD_INST_B=B (see ../build.py).
#include "pass_tma.cuh"

#if !defined(MVD_INST_A) || !defined(MVD_INST_B)
#error "compile with -DMVD_INST_A=<A> -DMVD_INST_B=<B>"
#endif

#define MVD_CAT_(a, b, c, d) a##b##c##d
#define MVD_CAT(a, b, c, d) MVD_CAT_(a, b, c, d)

namespace mvd {
extern const LengthOps MVD_CAT(ops_, MVD_INST_A, _, MVD_INST_B);
namespace {
using L = Launch<MVD_INST_A, MVD_INST_B>;
using LT = LaunchTma<MVD_INST_A, MVD_INST_B>;
cudaError_t init_all() {
  cudaError_t e = L::init();
  return e != cudaSuccess ? e : LT::init();
}
}  // namespace
const LengthOps MVD_CAT(ops_, MVD_INST_A, _, MVD_INST_B) = {
    L::Cfg::M, MVD_INST_A, MVD_INST_B, L::Cfg::MAX_THREADS, &init_all, &L::strided, &L::zconv, &L::xrow,
    &L::strided_smem, &L::xrow_smem, &LT::xrow, &LT::xrow_smem, &LT::xrow_blocks_per_sm, &LT::xrow_flags_of,
    &LT::strided, &LT::strided_smem, &LT::strided_blocks_per_sm, &LT::zconv, &LT::zconv_smem, &LT::zconv_blocks_per_sm};
}  // namespace mvd
