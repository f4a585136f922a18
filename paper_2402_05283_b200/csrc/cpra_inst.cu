// cpra_inst.cu -- compiled once per image size with -DCPRA_INST_N=<N>: the kernels and launch logic of that size.
#ifndef CPRA_INST_N
#error "compile with -DCPRA_INST_N=<N>"
#endif
#include "cpra_plan.cuh"

namespace cpra {
template struct Launch<CPRA_INST_N>;
}
