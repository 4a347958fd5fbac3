// sbf_inst_sweep.cu — the (s, m, H) cross product of BASELINE config 5 at k = 31 (Fig. 4): this ONE file is
// compiled once per (s, m) pair with -DSBF_SWEEP_S=<s> -DSBF_SWEEP_M=<m> (build.py), each object holding the five H
// instances of that pair.  Compiled without the two macros it is empty.
#include "sbf_dispatch.h"
#if defined(SBF_SWEEP_S) && defined(SBF_SWEEP_M)
namespace sbfk {
static const KernelEntry kTable[] = {
    SBF_ENTRY(31, SBF_SWEEP_M, SBF_SWEEP_S, 1),
    SBF_ENTRY(31, SBF_SWEEP_M, SBF_SWEEP_S, 2),
#if !(SBF_SWEEP_S == 28 && SBF_SWEEP_M == 16) // (28,16,4) is sbf_inst_default.cu
    SBF_ENTRY(31, SBF_SWEEP_M, SBF_SWEEP_S, 4),
#endif
    SBF_ENTRY(31, SBF_SWEEP_M, SBF_SWEEP_S, 6),
    SBF_ENTRY(31, SBF_SWEEP_M, SBF_SWEEP_S, 8),
};
static const TableRegistration kReg(kTable, (int)(sizeof(kTable) / sizeof(kTable[0])));
} // namespace sbfk
#endif
