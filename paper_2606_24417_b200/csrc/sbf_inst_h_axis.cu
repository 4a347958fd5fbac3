// sbf_inst_h_axis.cu — specialised stream_kernel instances (h_axis); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
    SBF_ENTRY(31, 16, 28, 1),
    SBF_ENTRY(31, 16, 28, 2),
    SBF_ENTRY(31, 16, 28, 6),
    SBF_ENTRY(31, 16, 28, 8),
};
const KernelEntry *inst_table_h_axis(int *n) { *n = (int)(sizeof(kTable) / sizeof(kTable[0])); return kTable; }
} // namespace sbfk
