// dpsr_kernels.cuh -- block bodies of the FFT / spectral-solve kernels of the DPSR path.
//
// Data layout in HBM (per batch item, per channel), H = N/2:
//   real grids      float  [N][N][N]            x slowest, z fastest (the C-ABI layout)
//   main spectrum   float2 [N][N][H]            slots (px, py, pz) in *stored order* on every axis
//   Nyquist plane   float2 [N][N]               the kz = N/2 column of every z-line, slots (px, py)
// "Stored order": slot p of an axis holds frequency pos2freq<len>(p) (fft_core.cuh); x and y are
// length-N complex transforms, z is a real transform done as an H-point complex FFT + split.
//
// Bodies are templates over a context (thread id, thread count, barrier) so the same source can be
// stepped on the host by a debugging harness; the library only instantiates them with DevCtx.
#pragma once
#include "fft_core.cuh"
#include "zy_pass.cuh"
#include "spectral.cuh"
