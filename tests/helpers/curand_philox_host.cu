// Test helper (third implementation for the Philox pin): runs cuRAND's own raw
// curand_Philox4x32_10(uint4, uint2) — the toolkit header's HOST code path — over counters read
// from a file.  Compiled by tests/test_oracle_rng.py with `nvcc` (host only; no GPU needed).
// usage: curand_philox_host <in: n*4 u32 counters> <out: n*4 u32> <key0> <key1>
#define QUALIFIERS static inline __host__ __device__
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <vector_types.h>
#include <curand_philox4x32_x.h>

int main(int argc, char** argv) {
  if (argc != 5) return 2;
  FILE* fi = fopen(argv[1], "rb");
  if (!fi) return 3;
  fseek(fi, 0, SEEK_END);
  long bytes = ftell(fi);
  fseek(fi, 0, SEEK_SET);
  std::vector<unsigned int> in(bytes / 4), out(bytes / 4);
  if (fread(in.data(), 4, in.size(), fi) != in.size()) return 4;
  fclose(fi);
  uint2 key = make_uint2((unsigned)strtoul(argv[3], 0, 10), (unsigned)strtoul(argv[4], 0, 10));
  for (size_t i = 0; i + 3 < in.size(); i += 4) {
    uint4 c = make_uint4(in[i], in[i + 1], in[i + 2], in[i + 3]);
    uint4 r = curand_Philox4x32_10(c, key);
    out[i] = r.x; out[i + 1] = r.y; out[i + 2] = r.z; out[i + 3] = r.w;
  }
  FILE* fo = fopen(argv[2], "wb");
  fwrite(out.data(), 4, out.size(), fo);
  fclose(fo);
  return 0;
}
