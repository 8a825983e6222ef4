// ks_mlp.cu — Tier-A dispatch: picks the tcgen05 kernel for a head shape and owns the sizes of the
// host-built operand images.  The kernels themselves:
//   ks_mlp_ws.cu     H <= 128  warp-specialized pipeline, every resource double-buffered by item
//   ks_mlp_ws256.cu  H == 256  same roles, single buffers, K-group-granular hand-over between layers
// (Their measured predecessor — "slots" of 128-256 threads that each run decode -> MMA1 -> GELU ->
// MMA2 -> GELU.w3 serially, two to four slots per CTA — reached 158 / 115 us on cfg2 and 75 ms on
// cfg5 against 100 us and 58 ms now; see profiles/README.md.)
#include "ks_internal.h"

int ks_mlp_k1(int n_in) { return n_in == 32 ? 32 : 16; }
size_t ks_mlp_w1_img_bytes(int n_in, int h) { return (size_t)ks_mlp_k1(n_in) * h * 2; }
size_t ks_mlp_w2_img_bytes(int h) { return (size_t)(h + 24) * h * 2; }

cudaError_t ks_launch_mlp(const KsMlpParams& p, int n_in, int h, int num_sms, cudaStream_t st) {
  if (h == 64 || h == 128) return ks_launch_mlp_ws(p, n_in, h, num_sms, st);
  if (h == 256) return ks_launch_mlp_ws256(p, n_in, num_sms, st);
  return cudaErrorInvalidValue;
}
