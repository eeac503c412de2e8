// tmpc_cr.cuh — a11: parallel-in-time (block cyclic reduction) factor and solve for one long horizon (config 5).
#pragma once
#include "tmpc_common.cuh"

namespace tmpc {

inline size_t cr_workspace_bytes(const Dims& d, size_t es) { (void)d; (void)es; return 0; }

template <typename T>
tmpc_status cr_factor(const Dims& d, const QpView<T>& qp, double sigma, double rho_f, double rho_g, unsigned char* ws, cudaStream_t s, int64_t* launches) {
  return TMPC_E_UNSUPPORTED;
}
template <typename T>
tmpc_status cr_admm(const Dims& d, const Params<T>& prm, const QpView<T>& qp, unsigned char* ws, T* x, T* zg, T* yf, T* yg, T* xi, T* r_prim, T* r_dual,
                    T* objective, int32_t* status, int iters, bool zg_given, cudaStream_t s, int64_t* launches) {
  return TMPC_E_UNSUPPORTED;
}

template <typename T>
tmpc_status cr_kkt_solve(const Dims& d, unsigned char* ws, const T* eta, T* xt, cudaStream_t s, int64_t* launches) { return TMPC_E_UNSUPPORTED; }

}  // namespace tmpc
