// dock_oracle_count.cpp -- the UNCHANGED oracle (dock_oracle.c) compiled with an operation-counting scalar in place
// of `double` (opcount.hpp).  TEST INFRASTRUCTURE; built by oracle.build_counted() into liboracle_count.so, which has the
// same C ABI as liboracle.so plus orc_count_reset / orc_count_get.  Used by bench.py's cpu_baseline leg to report the
// algorithmic flops of one evaluation.
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "opcount.hpp"

extern "C" {
uint64_t g_opcount[OC_N];
void orc_count_reset(void) { for (int k = 0; k < OC_N; ++k) g_opcount[k] = 0; }
void orc_count_get(uint64_t out[OC_N]) { for (int k = 0; k < OC_N; ++k) out[k] = g_opcount[k]; }
}

#undef isfinite
#define isfinite(x) oc_isfinite(x)
#define double cdouble
#include "dock_oracle.c"
