// bin_params.cuh -- the record the pair binning (k_bin.cu) reads per visible Gaussian, and the flat test space's chunk size.
// Shared by the two kernels that can write those records: k_scan_area (k_bin.cu) and the one-launch depth sort
// (k_sort.cu), whose last stage does k_scan_area's work.  Nothing here is decision arithmetic that could be contracted:
// kC / kA are single multiplications by a correctly rounded reciprocal.  NOT shared with oracle/.
#pragma once
#include "tgs_internal.cuh"

constexpr int BIN_THREADS = 128;
constexpr int BIN_IPT = 8;
constexpr int BIN_CHUNK = BIN_THREADS * BIN_IPT;      // tests per work item of k_bin

// Tile-test parameters of one visible Gaussian; 48 B, written in SORTED order by k_scan_area so that a k_bin chunk
// reads the parameters of its Gaussians as one contiguous, coalesced block instead of gathering three records each
// (scenes of many small Gaussians -- config 4: ~500 Gaussians per 1024-test chunk -- were bound by those gathers).
struct alignas(16) GaussParams {
  float u, v, A, B;
  float C, tau, kC, kA;                 // kC ~ -B/C, kA ~ -B/A
  uint32_t g, lo, w, pad;               // lo = x_lo | y_lo << 16
};
static_assert(sizeof(GaussParams) == 48, "three uint4 per Gaussian");

// from the 32-byte record k_preprocess writes for A5a (rec_bin: {u, v, A, B}, {C, tau, bits(trect.x), bits(trect.y)});
// *area = tests of the Gaussian
__device__ __forceinline__ GaussParams make_params_bin(uint32_t g, float4 r0, float4 r1, bool exact, uint32_t* area) {
  const uint32_t rx = __float_as_uint(r1.z), ry = __float_as_uint(r1.w);
  GaussParams P;
  P.g = g; P.lo = (rx & 0xffffu) | ((ry & 0xffffu) << 16); P.w = (rx >> 16) - (rx & 0xffffu); P.pad = 0;
  *area = P.w * ((ry >> 16) - (ry & 0xffffu));
  P.u = P.v = P.A = P.B = P.C = P.kC = P.kA = 0.0f; P.tau = 0.0f;
  if (exact) {
    P.u = r0.x; P.v = r0.y; P.A = r0.z; P.B = r0.w; P.C = r1.x; P.tau = r1.y;
    P.kC = -r0.w * __frcp_rn(r1.x); P.kA = -r0.w * __frcp_rn(r0.z);
  }
  return P;
}
__device__ __forceinline__ void store_params(uint4* __restrict__ dst, const GaussParams& P) {
  const uint4* s = reinterpret_cast<const uint4*>(&P);
  dst[0] = s[0]; dst[1] = s[1]; dst[2] = s[2];
}
__device__ __forceinline__ GaussParams load_params(const uint4* __restrict__ src) {
  GaussParams P;
  uint4* d = reinterpret_cast<uint4*>(&P);
  d[0] = src[0]; d[1] = src[1]; d[2] = src[2];
  return P;
}

