// Host-only check of the shared-memory plans of the resident kernel (tmpc_admm3.cuh): every plan terminates (the stride search is a loop), respects
// the alignments the kernel's vector accesses assume, and its byte count covers the records it places.  Built and run by tests/test_abi_and_host.py.
#include <cstdio>
#include "../paper_2606_24039_b200/csrc/tmpc_admm3.cuh"
using namespace tmpc;

static int fails = 0;
#define CHECK(c, ...) do { if (!(c)) { if (fails < 20) { printf("FAIL %s: ", #c); printf(__VA_ARGS__); printf("\n"); } ++fails; } } while (0)

template <typename T, int NC, int NX, bool XG>
void one(int Tn, int ng, int g_sel) {
  Dims d; memset(&d, 0, sizeof(d));
  d.T = Tn; d.N = Tn - 1; d.n = NC; d.nx = NX; d.nu = NC - NX; d.ng = ng; d.g_sel = g_sel; d.B = 4;
  using RC = Rec3<T, NC, NX, XG>;
  const int V = RC::V, w128 = 128 / (int)sizeof(T), m = Tn / 2;
  for (int pg = 1; pg <= (XG ? 1 : 2); ++pg) {
    const Admm3Plan P = admm3_plan<T, NC, NX, XG>(d, pg);
    const int need = ((g_sel || XG) ? RC::G : RC::G + RC::up(ng * NC));
    CHECK(P.R >= need, "T=%d ng=%d R=%d need=%d", Tn, ng, P.R, need);
    CHECK(P.R % (NC == 6 && sizeof(T) == 4 && !XG ? 2 : V) == 0, "stride alignment R=%d", P.R);
    CHECK(P.down0 % V == 0 && P.down0 % w128 == 64 / (int)sizeof(T), "down0=%d", P.down0);
    CHECK(P.down0 >= (m + 1) * P.R, "down0=%d overlaps the up half", P.down0);
    CHECK(P.per_problem >= P.down0 + (Tn - 1 - m) * P.R && P.per_problem % V == 0, "per_problem=%d", P.per_problem);
    CHECK((admm3_smem_bytes<T, NC, NX, XG>(d, pg) == (size_t)P.per_problem * pg * sizeof(T)), "bytes");
  }
  const Admm3Plan C = admm3_cl_plan<T, NC, NX, XG>(d);
  const int nrecs = (m + 1 > Tn - m) ? m + 1 : Tn - m;
  CHECK(C.down0 == 0 && C.per_problem >= nrecs * C.R + NC && C.per_problem % V == 0, "cluster plan per_problem=%d R=%d", C.per_problem, C.R);
  CHECK((C.per_problem * sizeof(T)) % 8 == 0, "mbarriers 8-byte aligned");
  CHECK((admm3_cl_smem_bytes<T, NC, NX, XG>(d) == (size_t)C.per_problem * sizeof(T) + 32), "cluster bytes");
}

template <typename T, int NC, int NX>
void shape() {
  for (int Tn = 2; Tn <= 700; ++Tn)
    for (int ng = 0; ng <= NC; ng += (NC > 6 ? 3 : 1))
      for (int g_sel = 0; g_sel <= 1; ++g_sel) { one<T, NC, NX, false>(Tn, ng, g_sel); one<T, NC, NX, true>(Tn, ng, g_sel); }
}

int main() {
  shape<float, 6, 4>(); shape<double, 6, 4>(); shape<float, 8, 6>(); shape<double, 8, 6>(); shape<float, 12, 8>(); shape<double, 12, 8>();
  // the two capacity claims of DESIGN.md 5.1: (64,160,8,4) fp64 fits one SM with the chain's share, (64,320,8,4) fp64 fits a pair
  Dims d; memset(&d, 0, sizeof(d)); d.n = 12; d.nx = 8; d.nu = 4; d.ng = 4; d.g_sel = 1; d.B = 64;
  d.T = 161; d.N = 160; { const size_t b1 = admm3_smem_bytes<double, 12, 8, true>(d, 1); CHECK(b1 <= 227u * 1024u, "N=160 chain share: %zu", b1); }
  d.T = 321; d.N = 320; { const size_t b2 = admm3_cl_smem_bytes<double, 12, 8, true>(d); CHECK(b2 <= 227u * 1024u, "N=320 pair: %zu", b2); }
  { const size_t b3 = admm3_smem_bytes<double, 12, 8, true>(d, 1); CHECK(b3 > 227u * 1024u, "N=320 must not fit one SM: %zu", b3); }
  printf(fails ? "plan_check: %d failures\n" : "plan_check: ok\n", fails);
  return fails ? 1 : 0;
}
