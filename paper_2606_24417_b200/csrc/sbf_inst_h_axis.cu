// sbf_inst_h_axis.cu — specialised stream_kernel instances (h_axis); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
#ifndef SBF_ONLY_DEFAULT // tuning builds compile the default instance only
    SBF_ENTRY(31, 16, 28, 1),
    SBF_ENTRY(31, 16, 28, 2),
    SBF_ENTRY(31, 16, 28, 6),
    SBF_ENTRY(31, 16, 28, 8),
#endif
    {0, 0, 0, 0, nullptr, nullptr, nullptr}, // terminator (not counted)
};
const KernelEntry *inst_table_h_axis(int *n) { *n = (int)(sizeof(kTable) / sizeof(kTable[0])) - 1; return kTable; }
} // namespace sbfk
