// tgs_ply.cu -- SURVEY 8(f) f4: loader for trained 3DGS checkpoints in the public `point_cloud.ply` layout the paper's
// scenes are stored in ("3DGS ... checkpoints", L55: mean, covariance from scale + rotation, opacity, SH).
// One vertex = a row of little-endian float32 properties named
//   x y z | nx ny nz (ignored) | f_dc_0..2 | f_rest_0..3(K-1)-1 (channel-major: index = ch (K-1) + (k-1)) |
//   opacity (logit) | scale_0..2 (log) | rot_0..3 (w x y z, not normalised)
// in any order; the header is parsed on the host (text), the rows are uploaded as they are, and k_ply_activate applies
// the activations on the device: scale = exp(raw), opacity = 1 / (1 + exp(-raw)), SH re-interleaved to [n][K][3].
// The result goes through the same tgs_load_gaussians(TGS_DEVICE) repack as every other scene.
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "tgs_internal.cuh"

namespace {

struct PlyLayout {
  int stride;            // floats per vertex
  int x, y, z, opacity;
  int scale[3], rot[4], dc[3];
  int rest0;             // offset of f_rest_0 (the f_rest_* properties must be consecutive and in order), -1 if none
  int K;                 // SH coefficients per channel
};

__global__ void __launch_bounds__(256) k_ply_activate(uint32_t n, PlyLayout L, const float* __restrict__ rows, float* __restrict__ means,
                                                      float* __restrict__ scales, float* __restrict__ quats, float* __restrict__ opacity,
                                                      float* __restrict__ sh, uint32_t* __restrict__ bad) {
  const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  const float* r = rows + (size_t)g * L.stride;
  bool ok = true;
  const float m[3] = {r[L.x], r[L.y], r[L.z]};
  for (int i = 0; i < 3; ++i) { means[3 * (size_t)g + i] = m[i]; ok = ok && isfinite(m[i]); }
  for (int i = 0; i < 3; ++i) { const float s = expf(r[L.scale[i]]); scales[3 * (size_t)g + i] = s; ok = ok && isfinite(s); }
  for (int i = 0; i < 4; ++i) { const float q = r[L.rot[i]]; quats[4 * (size_t)g + i] = q; ok = ok && isfinite(q); }
  const float o = 1.0f / (1.0f + expf(-r[L.opacity]));
  opacity[g] = o; ok = ok && isfinite(o);
  float* out = sh + (size_t)g * L.K * 3;
  for (int ch = 0; ch < 3; ++ch) {
    const float v = r[L.dc[ch]];
    out[ch] = v; ok = ok && isfinite(v);
    for (int k = 1; k < L.K; ++k) {
      const float w = r[L.rest0 + ch * (L.K - 1) + (k - 1)];
      out[k * 3 + ch] = w; ok = ok && isfinite(w);
    }
  }
  if (!ok) atomicAdd(bad, 1u);
}

}  // namespace

// implemented in tgs_api.cu (the context is opaque here)
extern "C" {
int tgs_ply_report(tgs_ctx* c, const char* msg);
cudaStream_t tgs_ply_stream(tgs_ctx* c);
int tgs_ply_device(tgs_ctx* c);
}

static int load_ply_impl(tgs_ctx* c, const char* path);

// No exception crosses the C-ABI: std::bad_alloc / std::length_error from the host-side containers become an error code.
extern "C" int tgs_load_ply(tgs_ctx* c, const char* path) {
  if (!c || !path) return TGS_E_INVALID_ARG;
  try {
    return load_ply_impl(c, path);
  } catch (...) {
    tgs_ply_report(c, "tgs_load_ply: out of host memory or malformed header");
    return TGS_E_INVALID_ARG;
  }
}

static int load_ply_impl(tgs_ctx* c, const char* path) {
  FILE* f = fopen(path, "rb");
  if (!f) { tgs_ply_report(c, "tgs_load_ply: cannot open file"); return TGS_E_INVALID_ARG; }
  struct FileGuard { FILE*& f; ~FileGuard() { if (f) fclose(f); } } guard{f};     // also on an exception
  auto bail = [&](const char* msg) { tgs_ply_report(c, msg); return (int)TGS_E_INVALID_ARG; };
  // ---- header
  char line[512];
  if (!fgets(line, sizeof(line), f) || strncmp(line, "ply", 3) != 0) return bail("tgs_load_ply: not a ply file");
  bool fmt_ok = false, in_vertex = false, done = false;
  unsigned long long n = 0;
  std::vector<std::string> props;
  while (fgets(line, sizeof(line), f)) {
    char a[64] = "", b[64] = "", d[64] = "";
    const int k = sscanf(line, "%63s %63s %63s", a, b, d);
    if (k >= 1 && !strcmp(a, "end_header")) { done = true; break; }
    if (k >= 3 && !strcmp(a, "format")) fmt_ok = !strcmp(b, "binary_little_endian");
    else if (k >= 3 && !strcmp(a, "element")) { in_vertex = !strcmp(b, "vertex"); if (in_vertex) n = strtoull(d, nullptr, 10); }
    else if (k >= 3 && !strcmp(a, "property") && in_vertex) {
      if (strcmp(b, "float") && strcmp(b, "float32")) return bail("tgs_load_ply: vertex properties must be float32");
      props.emplace_back(d);
    }
  }
  if (!done || !fmt_ok) return bail("tgs_load_ply: header incomplete or not binary_little_endian");
  if (n == 0 || n > 0xfffffff0ull) return bail("tgs_load_ply: bad vertex count");
  PlyLayout L;
  L.stride = (int)props.size();
  auto find = [&](const std::string& name) { for (size_t i = 0; i < props.size(); ++i) if (props[i] == name) return (int)i; return -1; };
  L.x = find("x"); L.y = find("y"); L.z = find("z"); L.opacity = find("opacity");
  for (int i = 0; i < 3; ++i) { L.scale[i] = find("scale_" + std::to_string(i)); L.dc[i] = find("f_dc_" + std::to_string(i)); }
  for (int i = 0; i < 4; ++i) L.rot[i] = find("rot_" + std::to_string(i));
  bool all = L.x >= 0 && L.y >= 0 && L.z >= 0 && L.opacity >= 0;
  for (int i = 0; i < 3; ++i) all = all && L.scale[i] >= 0 && L.dc[i] >= 0;
  for (int i = 0; i < 4; ++i) all = all && L.rot[i] >= 0;
  if (!all) return bail("tgs_load_ply: a required property is missing (x y z opacity scale_0..2 rot_0..3 f_dc_0..2)");
  int n_rest = 0;
  L.rest0 = find("f_rest_0");
  if (L.rest0 >= 0) while (find("f_rest_" + std::to_string(n_rest)) == L.rest0 + n_rest) ++n_rest;
  for (size_t i = 0; i < props.size(); ++i)
    if (props[i].rfind("f_rest_", 0) == 0 && ((int)i < L.rest0 || (int)i >= L.rest0 + n_rest)) return bail("tgs_load_ply: f_rest_* must be consecutive and in order");
  int deg = -1;
  for (int dgr = 0; dgr <= 3; ++dgr) if (3 * ((dgr + 1) * (dgr + 1) - 1) == n_rest) deg = dgr;
  if (deg < 0) return bail("tgs_load_ply: the number of f_rest_* properties fits no SH degree 0..3");
  L.K = (deg + 1) * (deg + 1);
  // ---- rows
  const size_t row_floats = (size_t)L.stride, total = row_floats * (size_t)n;
  {   // the header's vertex count is untrusted: compare it with what the file really holds before allocating anything
    const long data_at = ftell(f);
    if (data_at < 0 || fseek(f, 0, SEEK_END) != 0) return bail("tgs_load_ply: cannot seek");
    const long file_end = ftell(f);
    if (file_end < data_at || fseek(f, data_at, SEEK_SET) != 0) return bail("tgs_load_ply: cannot seek");
    if ((unsigned long long)(file_end - data_at) / sizeof(float) < (unsigned long long)total) return bail("tgs_load_ply: file shorter than the header says");
  }
  std::vector<float> rows(total);
  if (fread(rows.data(), sizeof(float), total, f) != total) return bail("tgs_load_ply: file shorter than the header says");
  fclose(f); f = nullptr;
  if (cudaSetDevice(tgs_ply_device(c)) != cudaSuccess) return TGS_E_CUDA;
  cudaStream_t s = tgs_ply_stream(c);
  float *d_rows = nullptr, *d_means = nullptr, *d_scales = nullptr, *d_quats = nullptr, *d_op = nullptr, *d_sh = nullptr;
  uint32_t* d_bad = nullptr;
  std::vector<void*> tmp;
  auto alloc = [&](void** p, size_t bytes) { if (cudaMalloc(p, bytes) != cudaSuccess) return false; tmp.push_back(*p); return true; };
  auto cleanup = [&]() { for (void* p : tmp) cudaFree(p); };
  const uint32_t N = (uint32_t)n;
  if (!alloc((void**)&d_rows, total * 4) || !alloc((void**)&d_means, (size_t)N * 12) || !alloc((void**)&d_scales, (size_t)N * 12) ||
      !alloc((void**)&d_quats, (size_t)N * 16) || !alloc((void**)&d_op, (size_t)N * 4) || !alloc((void**)&d_sh, (size_t)N * L.K * 12) ||
      !alloc((void**)&d_bad, 4)) { cleanup(); tgs_ply_report(c, "tgs_load_ply: out of device memory"); return TGS_E_CUDA; }
  uint32_t bad = 0;
  cudaMemcpyAsync(d_rows, rows.data(), total * 4, cudaMemcpyHostToDevice, s);
  cudaMemsetAsync(d_bad, 0, 4, s);
  k_ply_activate<<<(N + 255) / 256, 256, 0, s>>>(N, L, d_rows, d_means, d_scales, d_quats, d_op, d_sh, d_bad);
  cudaMemcpyAsync(&bad, d_bad, 4, cudaMemcpyDeviceToHost, s);
  if (cudaStreamSynchronize(s) != cudaSuccess || cudaGetLastError() != cudaSuccess) { cleanup(); tgs_ply_report(c, "tgs_load_ply: CUDA error"); return TGS_E_CUDA; }
  int rc = TGS_E_INVALID_ARG;
  if (bad) tgs_ply_report(c, "tgs_load_ply: non-finite value after activation");
  else rc = tgs_load_gaussians(c, N, deg, d_means, d_scales, d_quats, d_op, d_sh, TGS_DEVICE);
  cleanup();
  return rc;
}
