// sbf_inst_m_axis.cu — specialised stream_kernel instances (m_axis); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
#ifndef SBF_ONLY_DEFAULT // tuning builds compile the default instance only
    SBF_ENTRY(31, 12, 28, 4),
    SBF_ENTRY(31, 14, 28, 4),
    SBF_ENTRY(31, 18, 28, 4),
    SBF_ENTRY(31, 20, 28, 4),
#endif
    {0, 0, 0, 0, nullptr, nullptr, nullptr}, // terminator (not counted)
};
const KernelEntry *inst_table_m_axis(int *n) { *n = (int)(sizeof(kTable) / sizeof(kTable[0])) - 1; return kTable; }
} // namespace sbfk
