// lbmhd_inst.cu — instantiates every kernel of one (lattice, precision, scheme group); compiled once per triple with
//   -DLBMHD_INST_LAT=<1..5> -DLBMHD_INST_BITS=<64|32> -DLBMHD_INST_GROUP=<0|1>   (paper_2606_00641_b200/build.py runs these in
// parallel).  Group 0: IDEAL, INCRES, IDEAL_DIVB; group 1: RESIST, FULL.
#include "lbmhd_ops.cuh"

#if !defined(LBMHD_INST_LAT) || !defined(LBMHD_INST_BITS) || !defined(LBMHD_INST_GROUP)
#error "compile with -DLBMHD_INST_LAT=<lattice id> -DLBMHD_INST_BITS=<64|32> -DLBMHD_INST_GROUP=<0|1>"
#endif

#define LBH_CAT(lat, bits, grp) ops_table_##lat##_##bits##_g##grp
#define LBH_NAME(lat, bits, grp) LBH_CAT(lat, bits, grp)

namespace lbh {
#if LBMHD_INST_BITS == 64
OpTable LBH_NAME(LBMHD_INST_LAT, LBMHD_INST_BITS, LBMHD_INST_GROUP)(int scheme) { return table_for<LBMHD_INST_LAT, double, LBMHD_INST_GROUP>(scheme); }
#else
OpTable LBH_NAME(LBMHD_INST_LAT, LBMHD_INST_BITS, LBMHD_INST_GROUP)(int scheme) { return table_for<LBMHD_INST_LAT, float, LBMHD_INST_GROUP>(scheme); }
#endif
}  // namespace lbh
