// One instantiation of k_vn_pass per object file (compiled in parallel by build.py with -DVN_DV=.. -DVN_EXACT=..).
#include "vn_kernel.cuh"

#ifndef VN_DV
#error "compile with -DVN_DV=<register array size> -DVN_EXACT=<0|1>"
#endif

#define QC_CAT2(a, b) a##b
#define QC_CAT(a, b) QC_CAT2(a, b)

namespace qc {
void QC_CAT(launch_vn_dv, VN_DV)(const VnLaunch& L) { launch_vn<VN_DV, (VN_EXACT != 0)>(L); }
}  // namespace qc
