// sbf_inst_default.cu — the default configuration of the paper (k=31, m=16, s=28, H=4); see sbf_dispatch.h
#include "sbf_dispatch.h"
namespace sbfk {
static const KernelEntry kTable[] = {
    SBF_ENTRY(31, 16, 28, 4),
};
static const TableRegistration kReg(kTable, (int)(sizeof(kTable) / sizeof(kTable[0])));
} // namespace sbfk
