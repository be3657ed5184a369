// kr_codegen.h -- host side: validated network tables (KrHostNet) and the generator that turns them into the
// `struct KrNet` of constexpr tables which kr_spec.cuh is compiled against (NVRTC, at kr_network_create).
// Doubles are printed as hexadecimal floating literals, so the device sees the host's exact values.
#pragma once
#include <cstdio>
#include <string>
#include <vector>

#include "kr_tables.h"

struct KrHostNet {
  int E = 0, S = 0, R = 0, N = 0, energy = 0, n_aux = 0, any_rev = 0, any_tb = 0, any_qext = 0;
  double T_lo = 0, T_hi = 0, ln_p0_kB = 0;
  std::vector<int> sp, nu, flags, auxi, dnu_tot, comp, signed_row, row_ptr, col_ptr, row_ent, col_ent;
  std::vector<int> post_sp_ptr, post_sp_ent, post_res_ptr, post_res_ent, post_cmp_ptr, post_cmp_ent;   // kr_post.cuh lists
  std::vector<double> c0, A, beta, Ea, qk, tb, nasa, T_mid;
  // programs of the register-tile kernel (empty when N > 64)
  std::vector<KrDEnt> rprog;
  std::vector<int> rprog_ptr, fac, tgt, emeta[4];       // streams: [0..1] kr_wpc.cuh layout (32 / 64 threads), [2..3] kr_row.cuh layout
  int n_entries = 0, elen[4] = {0, 0, 0, 0};
  std::vector<KrETerm> estream[4];
  // balanced row program of kr_row.cuh (f rows and the T column): per group size (32 / 64 threads) a coalesced stream of
  // (reaction | (dnu + 128) << 16, partial-sum slot or -1) words and the slot range of every species
  std::vector<unsigned> rstream[2];
  std::vector<int> rslot_ptr[2];
  int rlen[2] = {0, 0}, n_rslots[2] = {0, 0};
  int row_compact = 0;           // 1: the row-layout term streams are in the compact two-factor form (see build_programs)
};

namespace kr_codegen {

inline std::string dbl(double x) {
  char b[64];
  if (x != x) return "(0.0/0.0)";
  if (x > 1.7976931348623157e308) return "(1.0/0.0)";
  if (x < -1.7976931348623157e308) return "(-1.0/0.0)";
  snprintf(b, sizeof b, "%a", x);
  return b;
}

template <class T, class F>
std::string arr1(const char* type, const char* name, const std::vector<T>& v, size_t n, F fmt) {
  std::string s = std::string("  static constexpr ") + type + " " + name + "[" + std::to_string(n ? n : 1) + "] = {";
  for (size_t i = 0; i < (n ? n : 1); ++i) { s += (i ? ", " : "") + (i < v.size() ? fmt(v[i]) : std::string("0")); }
  return s + "};\n";
}

template <class T, class F>
std::string arr2(const char* type, const char* name, const std::vector<T>& v, size_t n0, size_t n1, F fmt) {
  std::string s = std::string("  static constexpr ") + type + " " + name + "[" + std::to_string(n0 ? n0 : 1) + "][" +
                  std::to_string(n1) + "] = {";
  for (size_t i = 0; i < (n0 ? n0 : 1); ++i) {
    s += (i ? ",\n    {" : "\n    {");
    for (size_t j = 0; j < n1; ++j) {
      const size_t k = i * n1 + j;
      s += (j ? ", " : "") + (k < v.size() ? fmt(v[k]) : std::string("0"));
    }
    s += "}";
  }
  return s + "};\n";
}

// the translation unit handed to NVRTC: configuration macros, struct KrNet, then the kernel source
inline std::string net_header(const KrHostNet& H, int block, int min_blocks) {
  auto fi = [](int x) { return std::to_string(x); };
  auto fd = [](double x) { return dbl(x); };
  std::string s;
  s += "#define KRS_BLOCK " + std::to_string(block) + "\n#define KRS_MIN_BLOCKS " + std::to_string(min_blocks) + "\n";
  s += "struct KrNet {\n";
  s += "  static constexpr int E = " + fi(H.E) + ", S = " + fi(H.S) + ", R = " + fi(H.R) + ", N = " + fi(H.N) + ";\n";
  s += "  static constexpr int energy = " + fi(H.energy) + ", n_aux = " + fi(H.n_aux) + ", any_rev = " + fi(H.any_rev) +
       ", any_tb = " + fi(H.any_tb) + ", any_qext = " + fi(H.any_qext) + ";\n";
  s += "  static constexpr double T_lo = " + fd(H.T_lo) + ", T_hi = " + fd(H.T_hi) + ", ln_p0_kB = " + fd(H.ln_p0_kB) + ";\n";
  s += arr2("int", "sp", H.sp, H.R, 6, fi);
  s += arr2("int", "nu", H.nu, H.R, 6, fi);
  s += arr1("int", "flags", H.flags, H.R, fi);
  s += arr1("int", "auxi", H.auxi, H.R, fi);
  s += arr1("int", "dnu_tot", H.dnu_tot, H.R, fi);
  s += arr1("double", "c0", H.c0, H.R, fd);
  s += arr1("double", "A", H.A, H.R, fd);
  s += arr1("double", "beta", H.beta, H.R, fd);
  s += arr1("double", "Ea", H.Ea, H.R, fd);
  s += arr1("double", "qk", H.qk, H.R, fd);
  s += arr2("double", "tb_eff", H.tb, H.any_tb ? H.R : 1, H.S, fd);
  s += arr2("double", "nasa", H.nasa, H.S, 14, fd);
  s += arr1("double", "T_mid", H.T_mid, H.S, fd);
  s += arr2("int", "comp", H.comp, H.E, H.S, fi);
  s += arr1("int", "signed_row", H.signed_row, H.E, fi);
  s += arr1("int", "post_sp_ptr", H.post_sp_ptr, H.post_sp_ptr.size(), fi);
  s += arr1("int", "post_sp_ent", H.post_sp_ent, H.post_sp_ent.size(), fi);
  s += arr1("int", "post_res_ptr", H.post_res_ptr, H.post_res_ptr.size(), fi);
  s += arr1("int", "post_res_ent", H.post_res_ent, H.post_res_ent.size(), fi);
  s += arr1("int", "post_cmp_ptr", H.post_cmp_ptr, H.post_cmp_ptr.size(), fi);
  s += arr1("int", "post_cmp_ent", H.post_cmp_ent, H.post_cmp_ent.size(), fi);
  s += "};\n";
  return s;
}

}  // namespace kr_codegen
