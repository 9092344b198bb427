// vox.cu -- B200 (sm_100a) tetrahedral-mesh -> solid-binary-voxel hot path.
//
// Kernels:
//   K1 k1_count    per-tet voxel bbox -> tile range, sliver/degenerate cull, per-tile histogram
//   K2 k2_scan     exclusive scan of the tile counts (+ cursors, totals)
//   K3 k3_scatter  tet ids into per-tile lists
//   K4 k4_flat     one CTA per 32 x TY x TZ tile: exact integer edge functions of
//                  Theorem 1, one exact x-span per row, row words formed on
//                  chip, tile image stored once (no global atomics on the grid)
//   K5 (inside K4) large-tet path: exact tile classification + int64 span rows / 64-bit ballot rasteriser
//
// Exactness: inside(P) <=> four affine functions G_k(P) >= 0, each an exact integer
// (DESIGN.md "Arithmetic").  No floating point decides a bit.
#include "../../include/vox.h"

#include <cuda_runtime.h>
#include <pthread.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

// One translation unit, one libvox.so; the parts in include order (each .cuh is included exactly once, here):
#include "common.cuh"              // host context (Params, vox_ctx, workspace layout), check macros and the integer-geometry device helpers
#include "kernels_bin.cuh"         // the binning passes K1 (count), K2 (scan), K3 (scatter)
#include "kernel_tile.cuh"         // K4/K5 building blocks: planes, pair records, set-up paths, span arithmetic, row walk, tile epilogue
#include "kernel_lattice.cuh"      // K0 of the fused lattice path (vertex-plane slabs + packed vertex copy)
#include "kernel_tile_k4.cuh"      // the K4 kernel k4_flat (binned and fused-lattice instantiations)
#include "probe.cuh"               // vox_validate kernel and the integer-rate probe kernels
#include "api.cuh"                 // host side of the C ABI: create/tets/lattice/plan/run/status/noalloc/validate/run_host
#include "occupancy.cuh"           // the occupancy fold kernel and vox_occupancy
#include "pipe.cuh"                // vox_pipe_*: the transfer-overlapped pipeline
#include "api_misc.cuh"            // probe entry point, launch counter, checked-build status and self-test, error strings
