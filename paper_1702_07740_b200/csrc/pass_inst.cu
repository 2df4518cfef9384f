// One (DV, NG, EXACT) instantiation family of k_pass per object file (compiled in parallel by build.py with
// -DPASS_DV=.. -DPASS_NG=.. -DPASS_PCAP=.. -DPASS_EXACT=.. -DPASS_NAME=..).
#include "pass_kernel.cuh"

#if !defined(PASS_DV) || !defined(PASS_NG) || !defined(PASS_PCAP) || !defined(PASS_EXACT) || !defined(PASS_NAME)
#error "compile with -DPASS_DV=<column degree> -DPASS_NG=<gen edges per column> -DPASS_PCAP=<partner slots per gen edge> -DPASS_EXACT=<0|1> -DPASS_NAME=<symbol>"
#endif

namespace qc {
void PASS_NAME(const PassLaunch& L) { launch_pass<PASS_DV, PASS_NG, PASS_PCAP, (PASS_EXACT != 0)>(L); }
}  // namespace qc
