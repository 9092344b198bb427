// occupancy.cuh -- part of vox.cu (included there, once): the occupancy fold kernel and vox_occupancy.
#pragma once

// ------------------------------------------------------------------------------------------
// occupancy: k^3 sub-samples per voxel folded from the k-times finer bit grid (include/vox.h).  HBM bound:
// one thread reads the k*k fine words above one run of 32/k coarse voxels and writes 32/k bytes.
// ------------------------------------------------------------------------------------------
template <int K, int VEC>  // VEC fine words per thread and row (4: one 16-byte load per row)
__global__ void __launch_bounds__(256) k_occupancy(const u32* __restrict__ fine, int nx, int ny, int nz, int batch,
                                                   unsigned char* __restrict__ out) {
    constexpr int PER = 32 / K;                 // coarse voxels per fine word
    const int fw = (nx * K) >> 5;               // fine words per fine row
    const int fv = fw / VEC;
    const i64 total = (i64)batch * nz * ny * fv;
    const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int w = (int)(i % fv) * VEC;
    i64 rest = i / fv;
    const int y = (int)(rest % ny);
    rest /= ny;
    const int z = (int)(rest % nz);
    const i64 m = rest / nz;
    // SWAR: per fine word, K-bit group counts; even/odd groups accumulate in separate fields wide enough for K*K rows
    u32 A[VEC], B[VEC];
#pragma unroll
    for (int c = 0; c < VEC; ++c) A[c] = B[c] = 0;
    const i64 fny = (i64)ny * K, fnz = (i64)nz * K;
#pragma unroll
    for (int dz = 0; dz < K; ++dz)
#pragma unroll
        for (int dy = 0; dy < K; ++dy) {
            const u32* src = fine + ((m * fnz + (i64)z * K + dz) * fny + (i64)y * K + dy) * fw + w;
            u32 v[VEC];
            if (VEC == 4) {
                const uint4 q = __ldg(reinterpret_cast<const uint4*>(src));
                v[0] = q.x; v[1 % VEC] = q.y; v[2 % VEC] = q.z; v[3 % VEC] = q.w;
            } else {
                v[0] = __ldg(src);
            }
#pragma unroll
            for (int c = 0; c < VEC; ++c) {
                if (K == 2) {
                    const u32 s2 = (v[c] & 0x55555555u) + ((v[c] >> 1) & 0x55555555u);  // 16 fields of 2 bits: 0..2
                    A[c] += s2 & 0x33333333u;         // even voxels, 4-bit fields (sum <= 8)
                    B[c] += (s2 >> 2) & 0x33333333u;  // odd voxels
                } else {
                    const u32 s4 = v[c] - ((v[c] >> 1) & 0x77777777u) - ((v[c] >> 2) & 0x33333333u) - ((v[c] >> 3) & 0x11111111u);
                    A[c] += s4 & 0x0F0F0F0Fu;         // even voxels, byte fields (sum <= 64)
                    B[c] += (s4 >> 4) & 0x0F0F0F0Fu;  // odd voxels
                }
            }
        }
    unsigned char* dst = out + ((m * nz + z) * (i64)ny + y) * nx + (i64)w * PER;
#pragma unroll
    for (int c = 0; c < VEC; ++c) {
        if (K == 2) {
            u32 o[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {  // voxels 4q..4q+3 = A[2q], B[2q], A[2q+1], B[2q+1] (4-bit fields)
                const u32 a8 = (A[c] >> (8 * q)) & 0xFFu, b8 = (B[c] >> (8 * q)) & 0xFFu;
                o[q] = (a8 & 0xFu) | ((a8 & 0xF0u) << 12) | ((b8 & 0xFu) << 8) | ((b8 & 0xF0u) << 20);
            }
            *reinterpret_cast<uint4*>(dst + c * PER) = make_uint4(o[0], o[1], o[2], o[3]);
        } else {
            // voxels 0..7 = A0,B0,A1,B1 | A2,B2,A3,B3 (byte fields)
            *reinterpret_cast<uint2*>(dst + c * PER) = make_uint2(__byte_perm(A[c], B[c], 0x5140), __byte_perm(A[c], B[c], 0x7362));
        }
    }
}

extern "C" int vox_occupancy(void* cuda_stream, const uint32_t* d_bits_fine, int nx, int ny, int nz, int batch, int k,
                             uint8_t* d_counts_out) {
    if (!d_bits_fine || !d_counts_out || nx <= 0 || ny <= 0 || nz <= 0 || batch < 1) return VOX_EINVAL;
    if ((k != 2 && k != 4) || ((i64)nx * k) % 32 != 0) return VOX_EINVAL;
    if (((uintptr_t)d_counts_out & 15) != 0) return VOX_EINVAL;  // vector stores
    const int fw = (nx * k) >> 5;
    const bool vec = (fw % 4 == 0) && (((uintptr_t)d_bits_fine & 15) == 0);
    const i64 total = (i64)batch * nz * ny * (vec ? fw / 4 : fw);
    if (total > 0x7FFFFFFFll * 256) return VOX_ERANGE;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (k == 2 && vec) k_occupancy<2, 4><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    else if (k == 2) k_occupancy<2, 1><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    else if (vec) k_occupancy<4, 4><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    else k_occupancy<4, 1><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    return cudaGetLastError() == cudaSuccess ? VOX_OK : VOX_ECUDA;
}
