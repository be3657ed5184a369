// kr_jit.h -- host side: run-time compilation (NVRTC, sm_100a) and loading of the network-specialised kernel.
// NVRTC is dlopen'ed (no link-time dependency), the driver entry points come from cudaGetDriverEntryPoint, so
// the library still loads on a machine without a GPU.  Compiled cubins are cached in the process (per CUDA context) and
// on disk under a hash of the exact source and options: $KR_CACHE_DIR, else $XDG_CACHE_HOME/kratos_chem, else
// ~/.cache/kratos_chem, else /tmp/kratos_chem_cache_<uid>; the directory is created 0700 and must belong to the calling
// user, every file carries a length + checksum header that is verified before the image is used (a file that fails is
// ignored and recompiled).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <dlfcn.h>
#include <sys/stat.h>
#include <unistd.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

namespace kr_jit {

struct Kernel {
  CUmodule mod = nullptr;
  CUfunction fn = nullptr;
  int regs = 0, local_bytes = 0;
};

struct Driver {
  CUresult (*ModuleLoadData)(CUmodule*, const void*) = nullptr;
  CUresult (*ModuleGetFunction)(CUfunction*, CUmodule, const char*) = nullptr;
  CUresult (*FuncSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
  CUresult (*FuncGetAttribute)(int*, CUfunction_attribute, CUfunction) = nullptr;
  CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream,
                           void**, void**) = nullptr;
  CUresult (*OccupancyMaxActiveBlocksPerMultiprocessor)(int*, CUfunction, int, size_t) = nullptr;
  CUresult (*GetErrorString)(CUresult, const char**) = nullptr;
  CUresult (*CtxGetCurrent)(CUcontext*) = nullptr;
  bool ok = false;
};

inline Driver& driver() {
  static Driver d;
  static std::once_flag once;
  std::call_once(once, [] {
    auto get = [](const char* name, void** out) {
      cudaDriverEntryPointQueryResult q;
      return cudaGetDriverEntryPoint(name, out, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess && *out;
    };
    bool ok = true;
    ok &= get("cuModuleLoadData", (void**)&d.ModuleLoadData);
    ok &= get("cuModuleGetFunction", (void**)&d.ModuleGetFunction);
    ok &= get("cuFuncSetAttribute", (void**)&d.FuncSetAttribute);
    ok &= get("cuFuncGetAttribute", (void**)&d.FuncGetAttribute);
    ok &= get("cuLaunchKernel", (void**)&d.LaunchKernel);
    ok &= get("cuOccupancyMaxActiveBlocksPerMultiprocessor", (void**)&d.OccupancyMaxActiveBlocksPerMultiprocessor);
    ok &= get("cuGetErrorString", (void**)&d.GetErrorString);
    ok &= get("cuCtxGetCurrent", (void**)&d.CtxGetCurrent);
    cudaGetLastError();
    d.ok = ok;
  });
  return d;
}

// ---- NVRTC through dlopen ---------------------------------------------------------------------------------
struct Nvrtc {
  void* h = nullptr;
  int (*CreateProgram)(void**, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
  int (*CompileProgram)(void*, int, const char* const*) = nullptr;
  int (*GetProgramLogSize)(void*, size_t*) = nullptr;
  int (*GetProgramLog)(void*, char*) = nullptr;
  int (*GetCUBINSize)(void*, size_t*) = nullptr;
  int (*GetCUBIN)(void*, char*) = nullptr;
  int (*DestroyProgram)(void**) = nullptr;
  int (*Version)(int*, int*) = nullptr;
  bool ok = false;
  std::string where;
};

inline Nvrtc& nvrtc() {
  static Nvrtc n;
  static std::once_flag once;
  std::call_once(once, [] {
    std::vector<std::string> cands;
    if (const char* e = getenv("KR_NVRTC_LIB")) cands.push_back(e);
    cands.push_back("libnvrtc.so.12");
    cands.push_back("/usr/local/cuda/lib64/libnvrtc.so.12");
    cands.push_back("/usr/local/cuda/lib64/libnvrtc.so");
    cands.push_back("libnvrtc.so");
    for (const auto& c : cands) {
      n.h = dlopen(c.c_str(), RTLD_NOW | RTLD_LOCAL);
      if (n.h) { n.where = c; break; }
    }
    if (!n.h) return;
    bool ok = true;
    auto sym = [&](const char* name, void** out) { *out = dlsym(n.h, name); ok = ok && *out; };
    sym("nvrtcCreateProgram", (void**)&n.CreateProgram);
    sym("nvrtcCompileProgram", (void**)&n.CompileProgram);
    sym("nvrtcGetProgramLogSize", (void**)&n.GetProgramLogSize);
    sym("nvrtcGetProgramLog", (void**)&n.GetProgramLog);
    sym("nvrtcGetCUBINSize", (void**)&n.GetCUBINSize);
    sym("nvrtcGetCUBIN", (void**)&n.GetCUBIN);
    sym("nvrtcDestroyProgram", (void**)&n.DestroyProgram);
    sym("nvrtcVersion", (void**)&n.Version);
    n.ok = ok;
  });
  return n;
}

inline uint64_t fnv1a(const std::string& s, uint64_t h = 1469598103934665603ull) {
  for (unsigned char c : s) { h ^= c; h *= 1099511628211ull; }
  return h;
}

// "" when no directory that belongs to the calling user (and to nobody else) can be had: the disk cache is then off
inline std::string cache_dir() {
  std::string d;
  if (const char* e = getenv("KR_CACHE_DIR")) d = e;
  else if (const char* x = getenv("XDG_CACHE_HOME")) { d = std::string(x); mkdir(d.c_str(), 0700); d += "/kratos_chem"; }
  else if (const char* h = getenv("HOME")) { d = std::string(h) + "/.cache"; mkdir(d.c_str(), 0700); d += "/kratos_chem"; }
  else d = "/tmp/kratos_chem_cache_" + std::to_string((unsigned)getuid());
  mkdir(d.c_str(), 0700);
  struct stat st;
  if (stat(d.c_str(), &st) != 0 || !S_ISDIR(st.st_mode) || st.st_uid != getuid() || (st.st_mode & 022)) return "";
  return d;
}

struct CacheHeader { char magic[8]; uint64_t length, checksum; };

struct Header { const char* name; const char* text; };

// Compile `source` (with the given in-memory headers) for sm_100a.  Returns the cubin; on failure returns an
// empty vector and fills `log`.
inline std::vector<char> compile(const std::string& source, const std::vector<Header>& headers, std::string& log,
                                 bool* from_cache = nullptr) {
  std::vector<char> cubin;
  if (from_cache) *from_cache = false;
  Nvrtc& n = nvrtc();
  int vmaj = 0, vmin = 0;
  if (n.ok) n.Version(&vmaj, &vmin);
  std::string key = source;
  for (const auto& h : headers) { key += "\n//#"; key += h.name; key += "\n"; key += h.text; }
  key += "|sm_100a|c++17|lineinfo|nvrtc" + std::to_string(vmaj) + "." + std::to_string(vmin);
  char name[64];
  snprintf(name, sizeof name, "%016llx%016llx", (unsigned long long)fnv1a(key), (unsigned long long)fnv1a(key, 88172645463325252ull));
  const std::string dir = getenv("KR_NO_DISK_CACHE") ? std::string() : cache_dir();
  const std::string path = dir + "/" + name + ".krc";
  if (!dir.empty()) {
    if (FILE* f = fopen(path.c_str(), "rb")) {
      CacheHeader hd;
      if (fread(&hd, sizeof hd, 1, f) == 1 && std::string(hd.magic, 8) == "KRCUBIN1" && hd.length > 0 && hd.length < (1ull << 28)) {
        cubin.resize(size_t(hd.length));
        if (fread(cubin.data(), 1, cubin.size(), f) != cubin.size() ||
            fnv1a(std::string(cubin.begin(), cubin.end())) != hd.checksum)
          cubin.clear();                       // truncated or altered: recompile
      }
      fclose(f);
      if (!cubin.empty()) { if (from_cache) *from_cache = true; return cubin; }
    }
  }
  if (!n.ok) { log = "NVRTC not found (tried libnvrtc.so.12, /usr/local/cuda/lib64; set KR_NVRTC_LIB)"; return cubin; }
  std::vector<const char*> hn, ht;
  for (const auto& h : headers) { hn.push_back(h.name); ht.push_back(h.text); }
  void* prog = nullptr;
  const std::string pname = std::string("kr_spec_") + name + ".cu";
  if (n.CreateProgram(&prog, source.c_str(), pname.c_str(), int(headers.size()), ht.data(), hn.data()) != 0) {
    log = "nvrtcCreateProgram failed";
    return cubin;
  }
  const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo", "-default-device"};
  const int rc = n.CompileProgram(prog, 4, opts);
  size_t lsz = 0;
  n.GetProgramLogSize(prog, &lsz);
  if (lsz > 1) { log.resize(lsz); n.GetProgramLog(prog, &log[0]); }
  if (rc == 0) {
    size_t sz = 0;
    if (n.GetCUBINSize(prog, &sz) == 0 && sz > 0) {
      cubin.resize(sz);
      if (n.GetCUBIN(prog, cubin.data()) != 0) cubin.clear();
    }
  }
  n.DestroyProgram(&prog);
  if (!cubin.empty() && !dir.empty()) {
    const std::string tmp = path + "." + std::to_string(getpid()) + ".tmp";
    if (FILE* f = fopen(tmp.c_str(), "wb")) {
      CacheHeader hd;
      memcpy(hd.magic, "KRCUBIN1", 8);
      hd.length = cubin.size(); hd.checksum = fnv1a(std::string(cubin.begin(), cubin.end()));
      const bool ok = fwrite(&hd, sizeof hd, 1, f) == 1 && fwrite(cubin.data(), 1, cubin.size(), f) == cubin.size();
      fclose(f);
      if (ok) rename(tmp.c_str(), path.c_str()); else remove(tmp.c_str());
    }
  }
  return cubin;
}

// in-process cache: (CUDA context, cubin hash) -> loaded kernel (modules live until process exit)
inline bool load(const std::vector<char>& cubin, const char* entry, Kernel& out, std::string& err) {
  static std::mutex mu;
  static std::map<std::pair<uintptr_t, uint64_t>, Kernel> loaded;
  Driver& d = driver();
  if (!d.ok) { err = "CUDA driver entry points unavailable"; return false; }
  cudaFree(0);                                    // make sure the primary context of the current device is current
  CUcontext ctx = nullptr;
  if (d.CtxGetCurrent) d.CtxGetCurrent(&ctx);
  const std::pair<uintptr_t, uint64_t> key(reinterpret_cast<uintptr_t>(ctx), fnv1a(std::string(cubin.begin(), cubin.end())));
  std::lock_guard<std::mutex> lk(mu);
  auto it = loaded.find(key);
  if (it != loaded.end()) { out = it->second; return true; }
  Kernel k;
  CUresult r = d.ModuleLoadData(&k.mod, cubin.data());
  if (r == CUDA_SUCCESS) r = d.ModuleGetFunction(&k.fn, k.mod, entry);
  if (r != CUDA_SUCCESS) {
    const char* s = nullptr;
    d.GetErrorString(r, &s);
    err = std::string("loading the specialised kernel failed: ") + (s ? s : "?");
    return false;
  }
  d.FuncGetAttribute(&k.regs, CU_FUNC_ATTRIBUTE_NUM_REGS, k.fn);
  d.FuncGetAttribute(&k.local_bytes, CU_FUNC_ATTRIBUTE_LOCAL_SIZE_BYTES, k.fn);
  loaded[key] = k;
  out = k;
  return true;
}

}  // namespace kr_jit
