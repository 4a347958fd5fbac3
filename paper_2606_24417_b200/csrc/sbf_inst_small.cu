// sbf_inst_small.cu — specialised stream_kernel instances (small); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
#ifndef SBF_ONLY_DEFAULT // tuning builds compile the default instance only
    SBF_ENTRY(9, 5, 6, 4),
    SBF_ENTRY(32, 16, 28, 4),
    SBF_ENTRY(21, 11, 21, 3),
    SBF_ENTRY(15, 15, 12, 5),
#endif
    {0, 0, 0, 0, nullptr, nullptr, nullptr}, // terminator (not counted)
};
const KernelEntry *inst_table_small(int *n) { *n = (int)(sizeof(kTable) / sizeof(kTable[0])) - 1; return kTable; }
} // namespace sbfk
