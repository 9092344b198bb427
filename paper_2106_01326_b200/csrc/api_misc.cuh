// api_misc.cuh -- part of vox.cu (included there, once): probe entry point, launch counter, checked-build status and self-test, error strings.
#pragma once

extern "C" int vox_probe_int32(void* cuda_stream, int kind, int blocks, int iters, uint32_t* d_sink, double* ops_out) {
    if (blocks <= 0 || iters <= 0 || !d_sink) return VOX_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (kind == 0) k_probe<0><<<blocks, 256, 0, st>>>(iters, d_sink), count_launch();
    else if (kind == 1) k_probe<1><<<blocks, 256, 0, st>>>(iters, d_sink), count_launch();
    else k_probe<2><<<blocks, 256, 0, st>>>(iters, d_sink), count_launch();
    if (cudaGetLastError() != cudaSuccess) return VOX_ECUDA;
    if (ops_out) *ops_out = (double)blocks * 256.0 * (double)iters * 64.0;
    return VOX_OK;
}

extern "C" uint64_t vox_kernel_launches(void) { return __atomic_load_n(&g_launches, __ATOMIC_RELAXED); }

extern "C" int vox_debug_check_status(uint32_t* code_out) {
#ifdef VOX_CHECKS
    unsigned int c = 0, zero = 0;
    if (cudaDeviceSynchronize() != cudaSuccess) return VOX_ECUDA;
    if (cudaMemcpyFromSymbol(&c, g_check, sizeof(c)) != cudaSuccess) return VOX_ECUDA;
    if (cudaMemcpyToSymbol(g_check, &zero, sizeof(zero)) != cudaSuccess) return VOX_ECUDA;
    if (code_out) *code_out = c;
    return 1;
#else
    if (code_out) *code_out = 0;
    return 0;
#endif
}

// Operand-level self-test of the integer helpers of the row walk (checked build only; include/vox.h).  One thread per
// element; the helpers are the very functions K4 inlines.
#ifdef VOX_CHECKS
__global__ void __launch_bounds__(256) k_selftest(int op, const i64* __restrict__ a, const i64* __restrict__ b, i64 n,
                                                  int* __restrict__ out) {
    const i64 i = (i64)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const i64 x = a[i], y = b[i];
    int r = 0;
    if (op == 0) r = span_bound((int)x, -(int)(u32)y, recip_up((u32)y));
    else if (op == 1) r = span_bound((int)x, -(int)(u32)y, (int)(0xFFFFFFFFu / (u32)y + 1u));
    else if (op == 2) r = (int)(((u32)x * (u32)div_magic((int)y)) >> 16);
    else if (op == 3) r = span64_bound(x, y);
    else if (op == 4) r = recip_up((u32)y);
    out[i] = r;
}
#endif
extern "C" int vox_debug_selftest(void* cuda_stream, int op, const int64_t* d_a, const int64_t* d_b, int64_t n,
                                  int32_t* d_out) {
#ifdef VOX_CHECKS
    if (op < 0 || op > 4 || n < 0 || (n > 0 && (!d_a || !d_b || !d_out))) return VOX_EINVAL;
    if (n == 0) return 1;
    k_selftest<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(op, (const i64*)d_a, (const i64*)d_b, n, d_out);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? 1 : VOX_ECUDA;
#else
    (void)cuda_stream; (void)op; (void)d_a; (void)d_b; (void)n; (void)d_out;
    return 0;
#endif
}

extern "C" const char* vox_strerror(int code) {
    switch (code) {
        case VOX_OK: return "ok";
        case VOX_EINVAL: return "invalid argument";
        case VOX_ERANGE: return "argument out of the supported range";
        case VOX_EWORKSPACE: return "workspace too small";
        case VOX_ECUDA: return "CUDA runtime error (see vox_last_error)";
        case VOX_ESTATE: return "call order violated";
        case VOX_EDATA: return "mesh data out of range";
        default: return "unknown error";
    }
}

extern "C" const char* vox_last_error(const vox_ctx* ctx) { return ctx ? ctx->err : ""; }
