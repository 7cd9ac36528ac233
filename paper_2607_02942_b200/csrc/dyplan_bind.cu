// dyplan_bind.cu -- K_bind: coefficient construction, Algorithm 1 l.1-8 and Eq.(2).
// One thread per node: v_n = Psi(role, skill, fan-in) and, for each of the node's options, q = Q^(skill, model, policy),
// tau = sum over stages of the longest call's tokens / decode rate + prefill correction, c = total tokens / norm.
// fp64 with explicit rounding (no contraction), so the integer durations are reproducible bit for bit.
#include "dyplan_internal.cuh"

namespace dyplan {

__global__ void __launch_bounds__(128) k_bind(BindArgs a) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= a.NN) return;
  const dyplan_profiles& p = a.prof;
  const int s = a.skill[n], ro = a.role[n];
  const int fan = __popc(a.pred_mask[n]);
  const bool node_ok = s < p.S && ro < p.ROLES;
  a.vuln[n] = node_ok ? p.psi[((size_t)ro * p.S + s) * p.F + (fan < p.F - 1 ? fan : p.F - 1)] : __int_as_float(0x7fc00000);
  const int o0 = a.opt_off[n], o1 = a.opt_off[n + 1];
  for (int o = o0; o < o1 && o < a.KK; o++) {
    if (o < 0) continue;
    const int m = a.model[o], d = a.backend[o], pl = a.policy[o];
    const bool ok = node_ok && m < p.M && d < p.D && pl < p.P && p.theta_dec[m * p.D + d] > 0.0f;
    if (!ok) {
      a.acc[o] = __int_as_float(0x7fc00000); a.lat_us[o] = -1; a.cost[o] = __int_as_float(0x7fc00000);
      if (a.demand) a.demand[o] = -1;
      continue;
    }
    const size_t pair = ((size_t)s * p.M + m) * p.P + pl;
    const float* g = p.tokens + pair * p.A * p.J;
    double serial = 0.0, total = 0.0;
    for (int st = 0; st < p.A; st++) {
      double mx = 0.0;
      for (int j = 0; j < p.J; j++) {
        const double t = (double)g[st * p.J + j];
        mx = t > mx ? t : mx;              // "each parallel stage contributes its longest nominal call duration"
        total = __dadd_rn(total, t);       // "call cost sums all calls"
      }
      serial = __dadd_rn(serial, mx);      // "serial stage durations add"
    }
    const double tau = __dadd_rn(__ddiv_rn(__dmul_rn(1e6, serial), (double)p.theta_dec[m * p.D + d]), (double)p.tau_pre_us[m * p.D + d]);
    const double tr = rint(tau);
    a.acc[o] = p.quality[pair];
    a.lat_us[o] = (tr >= 0.0 && tr <= 2147483647.0) ? (int)tr : -1;
    a.cost[o] = (float)__ddiv_rn(total, (double)p.token_norm);
    if (a.demand) { const double dr = rint(total); a.demand[o] = (dr >= 0.0 && dr <= 2147483647.0) ? (int)dr : -1; }
  }
}

cudaError_t launch_bind(const BindArgs& a, cudaStream_t s) {
  if (a.NN <= 0) return cudaSuccess;
  k_bind<<<(unsigned)((a.NN + 127) / 128), 128, 0, s>>>(a);
  return cudaGetLastError();
}

}  // namespace dyplan
