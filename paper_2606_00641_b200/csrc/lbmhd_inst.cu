// lbmhd_inst.cu — instantiates every kernel of one (lattice, precision) pair; compiled once per pair with
//   -DLBMHD_INST_LAT=<1..5> -DLBMHD_INST_BITS=<64|32>   (paper_2606_00641_b200/build.py runs these in parallel).
#include "lbmhd_ops.cuh"

#if !defined(LBMHD_INST_LAT) || !defined(LBMHD_INST_BITS)
#error "compile with -DLBMHD_INST_LAT=<lattice id> -DLBMHD_INST_BITS=<64|32>"
#endif

#define LBH_CAT(lat, bits) ops_table_##lat##_##bits
#define LBH_NAME(lat, bits) LBH_CAT(lat, bits)

namespace lbh {
#if LBMHD_INST_BITS == 64
OpTable LBH_NAME(LBMHD_INST_LAT, LBMHD_INST_BITS)(int scheme) { return table_for<LBMHD_INST_LAT, double>(scheme); }
#else
OpTable LBH_NAME(LBMHD_INST_LAT, LBMHD_INST_BITS)(int scheme) { return table_for<LBMHD_INST_LAT, float>(scheme); }
#endif
}  // namespace lbh
