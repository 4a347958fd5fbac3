// sbf_inst_default.cu — specialised stream_kernel instances (default); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
    SBF_ENTRY(31, 16, 28, 4),
};
const KernelEntry *inst_table_default(int *n) { *n = (int)(sizeof(kTable) / sizeof(kTable[0])); return kTable; }
} // namespace sbfk
