// Minimal stand-alone form of the normative per-candidate arithmetic (O-2) for counting the SASS
// instructions one vote costs when written plainly ("I_fp32 = FP32-pipe SASS instructions
// of a minimal stand-alone O-2 device function").  NOT part of libhough_b200.so and never launched: it is
// compiled to a cubin by tests/test_abi_and_host.py::test_o2_instruction_count, which counts the floating-point
// instructions between the markers and checks them against the numbers bench.py's roofline uses
// (profiles/r02_o2_sass_count.md holds the listing).
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 --fmad=false -prec-div=true -ftz=false -cubin o2_count.cu
#include <stdint.h>

// per (hit, phi0 column): s = sin(phi - phi0c) and, in 3D, r*s and r^2 -- shared by the d0 bins of the column
// per (hit, d0 bin, phi0 column) = per candidate: the rest
extern "C" __global__ void o2_vote_3d(const float4* __restrict__ hit, const float* __restrict__ c0,
                                      const float* __restrict__ s0, const float* __restrict__ d0c,
                                      const float* __restrict__ two_d0, const float* __restrict__ d0sq, float kmax,
                                      float inv_dk, float nk_f, int* __restrict__ bin)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const float4 h = hit[i];                                    // {sin phi, cos phi, r, -}
    const float m1 = __fmul_rn(h.x, c0[i]);
    const float m2 = __fmul_rn(h.y, s0[i]);
    const float s = __fsub_rn(m1, m2);
    const float rs = __fmul_rn(h.z, s);
    const float r2 = __fmul_rn(h.z, h.z);
    const float t = __fadd_rn(rs, d0c[i]);
    const float num = __fadd_rn(t, t);
    const float a = __fmul_rn(two_d0[i], rs);
    const float b = __fadd_rn(r2, a);
    const float den = __fadd_rn(b, d0sq[i]);
    const float kappa = __fdiv_rn(num, den);
    const float v = __fadd_rn(kappa, kmax);
    const float u = __fmul_rn(v, inv_dk);
    bin[i] = (u >= 0.0f && u < nk_f) ? (int)u : -1;
}

extern "C" __global__ void o2_vote_2d(const float4* __restrict__ hit, const float* __restrict__ c0,
                                      const float* __restrict__ s0, float kmax, float inv_dk, float nk_f,
                                      int* __restrict__ bin)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const float4 h = hit[i];
    const float m1 = __fmul_rn(h.x, c0[i]);
    const float m2 = __fmul_rn(h.y, s0[i]);
    const float s = __fsub_rn(m1, m2);
    const float kappa = __fdiv_rn(__fadd_rn(s, s), h.z);
    const float v = __fadd_rn(kappa, kmax);
    const float u = __fmul_rn(v, inv_dk);
    bin[i] = (u >= 0.0f && u < nk_f) ? (int)u : -1;
}
