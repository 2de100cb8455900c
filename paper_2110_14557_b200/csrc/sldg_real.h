// sldg_real.h -- the storage / sweep-arithmetic type of the advection kernels.  Every sweep kernel file is compiled
// twice: as is (real = double, launchers suffixed _f64) and with -DSLDG_REAL_FLOAT (real = float, launchers suffixed
// _f32; single precision mode, reading W).  Shift decisions, rho, E and the field solve are fp64 in both.
#pragma once

#ifdef SLDG_REAL_FLOAT
typedef float real;
typedef float2 real2;
#define SLDG_SFX(name) name##_f32
__device__ __forceinline__ real2 make_real2(real a, real b) { return make_float2(a, b); }
#else
typedef double real;
typedef double2 real2;
#define SLDG_SFX(name) name##_f64
__device__ __forceinline__ real2 make_real2(real a, real b) { return make_double2(a, b); }
#endif
