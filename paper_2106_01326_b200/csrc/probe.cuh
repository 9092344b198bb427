// probe.cuh -- part of vox.cu (included there, once): vox_validate kernel and the integer-rate probe kernels.
#pragma once

// ------------------------------------------------------------------------------------------
// validation and probes
// ------------------------------------------------------------------------------------------
__global__ void k_validate(Params p, u32* hdr) {
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (i < p.V) {
        int x = p.verts[3 * i], y = p.verts[3 * i + 1], z = p.verts[3 * i + 2];
        bad = bad || x < 0 || x > p.ex || y < 0 || y > p.ey || z < 0 || z > p.ez;
    }
    if (i < p.T && !p.lcx) {
        int4 id = p.tets[i];
        bad = bad || id.x < 0 || id.x >= p.V || id.y < 0 || id.y >= p.V || id.z < 0 || id.z >= p.V || id.w < 0 || id.w >= p.V;
    }
    if (p.off && i <= p.batch) {
        i64 o = p.off[i];
        if (i == 0) bad = bad || (o != 0);
        if (i == p.batch) bad = bad || (o != p.T);
        if (i > 0) bad = bad || (o < p.off[i - 1]);
    }
    if (bad) hdr[H_BAD] = 1;
}

// dependent-free integer streams: 8 independent chains per thread
template <int KIND>
__global__ void __launch_bounds__(256) k_probe(int iters, u32* sink) {
    u32 a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    u32 b = blockIdx.x * 2654435761u + 12345u, c = b ^ 0x9E3779B9u;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (KIND == 0) {  // LOP3 only: alu pipe
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a0) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a1) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a2) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a3) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a4) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a5) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a6) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a7) : "r"(b), "r"(c));
            } else if (KIND == 1) {  // IMAD only: fma pipe
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a0) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a1) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a2) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a3) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a4) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a5) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a6) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a7) : "r"(b), "r"(c));
            } else {  // mixed: 4 LOP3 + 4 IMAD
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a0) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a1) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a2) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a3) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a4) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a5) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a6) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a7) : "r"(b), "r"(c));
            }
        }
    }
    u32 r = a0 ^ a1 ^ a2 ^ a3 ^ a4 ^ a5 ^ a6 ^ a7;
    if (r == 0x12345678u) sink[0] = r;  // practically never: keeps the chains alive
}
