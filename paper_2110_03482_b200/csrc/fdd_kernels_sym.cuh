// Step a4, symmetric kernel (stub: not built yet -- every plan falls back to the generic kernel).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace fdd {

struct SymTables {
    int dummy = 0;
};

inline int sym_build_tables(SymTables*, const double*, int, int, long long, bool* ok, size_t*)
{
    *ok = false;
    return 0;
}
inline void sym_free_tables(SymTables*) {}
inline int sym_launch(const SymTables&, const float2*, long long, int, long long, int, int, int,
                      float2*, long long, float, int, cudaStream_t)
{
    return -5;
}

}  // namespace fdd
