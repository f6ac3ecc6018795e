// prefill_umma.cu -- tcgen05 UMMA prefill (placeholder until the kernel lands: reports "not supported",
// so bf16 prefill runs on the SIMT tiles).
#include "common.cuh"

namespace jetlong {

bool umma_prefill_supported(long long, int, int, int, int) { return false; }
size_t umma_prefill_workspace_bytes(long long, int, int, int) { return 0; }
int launch_prefill_umma(const void*, const void*, const void*, void*, float*, long long, int, int, int, long long,
                        long long, double, bool, void*, size_t, cudaStream_t) {
    return JETLONG_UNSUPPORTED;
}

}  // namespace jetlong
