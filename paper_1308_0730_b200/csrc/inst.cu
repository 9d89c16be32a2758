// One translation unit per supported pencil length: compiled once for every MVD_LEN(A, B) line of
// lengths.def with -DMVD_INST_A=A -DMVD_INST_B=B (see ../build.py).
#include "pass_kernels.cuh"

#if !defined(MVD_INST_A) || !defined(MVD_INST_B)
#error "compile with -DMVD_INST_A=<A> -DMVD_INST_B=<B>"
#endif

#define MVD_CAT_(a, b, c, d) a##b##c##d
#define MVD_CAT(a, b, c, d) MVD_CAT_(a, b, c, d)

namespace mvd {
extern const LengthOps MVD_CAT(ops_, MVD_INST_A, _, MVD_INST_B);
const LengthOps MVD_CAT(ops_, MVD_INST_A, _, MVD_INST_B) = Launch<MVD_INST_A, MVD_INST_B>::ops();
}  // namespace mvd
