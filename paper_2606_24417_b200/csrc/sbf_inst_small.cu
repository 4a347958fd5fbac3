// sbf_inst_small.cu — a few other-k instances (worked example of Fig. 2, k = 32, odd shapes); see sbf_dispatch.h
#include "sbf_dispatch.h"
#ifndef SBF_ONLY_DEFAULT // tuning builds compile the default instance only
namespace sbfk {
static const KernelEntry kTable[] = {
    SBF_ENTRY(9, 5, 6, 4),
    SBF_ENTRY(32, 16, 28, 4),
    SBF_ENTRY(21, 11, 21, 3),
    SBF_ENTRY(15, 15, 12, 5),
};
static const TableRegistration kReg(kTable, (int)(sizeof(kTable) / sizeof(kTable[0])));
} // namespace sbfk
#endif
