// sbf_inst_s_axis.cu — specialised stream_kernel instances (s_axis); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
#ifndef SBF_ONLY_DEFAULT // tuning builds compile the default instance only
    SBF_ENTRY(31, 16, 24, 4),
    SBF_ENTRY(31, 16, 26, 4),
    SBF_ENTRY(31, 16, 30, 4),
    SBF_ENTRY(31, 16, 31, 4),
#endif
    {0, 0, 0, 0, nullptr, nullptr, nullptr}, // terminator (not counted)
};
const KernelEntry *inst_table_s_axis(int *n) { *n = (int)(sizeof(kTable) / sizeof(kTable[0])) - 1; return kTable; }
} // namespace sbfk
