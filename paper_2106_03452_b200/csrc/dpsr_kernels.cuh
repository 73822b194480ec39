// dpsr_kernels.cuh -- the FFT / spectral-solve kernels of the DPSR path.
//
// Data layout in HBM (per batch item, per channel), H = N/2:
//   real grids      float  [N][N][N]            x slowest, z fastest (the C-ABI layout)
//   main spectrum   float2 [N][N][H]            slots (px, py, pz) in *stored order* on every axis, the z slot
//                                               of line (x, y) kept in column pz ^ (y & 15) (kz_swz)
//   Nyquist plane   float2 [N][N]               the kz = N/2 column of every z-line, slots (px, py);
//                                               N >= 256 also keeps a transposed copy [py][px] between passes
// "Stored order": slot p of an axis holds frequency pos2freq<len>(p) (fft_core.cuh); x and y are
// length-N complex transforms, z is a real transform done as an H-point complex FFT + split.
//
//   zy_pass.cuh     splat + forward z + y pass of the fused planes (N <= 128), one plane per CTA
//   zwarp_pass.cuh  splat / Gbar' + forward z pass for N >= 256, one tile of 32 lines per CTA, a warp owns its lines
//   zwarp_inv.cuh   inverse z pass for N >= 256, the mirror of zwarp_pass.cuh
//   zline_pass.cuh  persistent bulk-copy z (+ y) passes: inverse, fused Gbar'
//   ring_pass.cuh   persistent TMA ring: x pass with the fused spectral solve / its adjoint, y pass (N >= 256)
#pragma once
#include "fft_core.cuh"
#include "spectral.cuh"
#include "zy_pass.cuh"
#include "zwarp_pass.cuh"
#include "ring_pass.cuh"
#include "zline_pass.cuh"
#include "zwarp_inv.cuh"
