// a6: block-sparse CSR variant of a2-a4 (placeholder until the dense path is measured).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <cstdio>
#include "../../include/dode.h"
#include "kernels_dense.cuh"

namespace dode {

struct CsrStore {
    bool ready = false;
};

inline void csr_forward(const CsrStore&, int, int, const float*, size_t, const float*, float*, int, const DayList&,
                        const dode_dims&, int, cudaStream_t, int64_t*) {}
inline void csr_gradient(const CsrStore&, int, int, const float*, float*, size_t, float*, float, int, const DayList&,
                         const dode_dims&, int, cudaStream_t, int64_t*) {}
inline void csr_free(CsrStore&) {}
inline int csr_build(CsrStore&, const dode_dims&, const dode_dar&, cudaStream_t, char* err) {
    snprintf(err, 512, "CSR storage is not built yet");
    return DODE_EINVAL;
}

}  // namespace dode
