// jit.h -- run-time specialisation of a kernel to one model: NVRTC compiles a CUDA source (a generated prelude of
// compile-time tables + a kernel file of this directory, embedded in the library at build time) to an sm_100a cubin, the
// CUDA runtime loads it (cudaLibraryLoadData) and hands back a cudaKernel_t that is launched like any other kernel.
// Compiled kernels are cached per process by the text of their prelude: handles of the same model share one compilation.
// NVRTC is opened with dlopen on first use, so the library itself loads on a machine without it (and without a GPU); a
// kernel that cannot be compiled is an error of tddp4_create -- there is no other code path.
#pragma once
#include <cuda_runtime.h>
#include <dlfcn.h>

#include <map>
#include <mutex>
#include <string>
#include <vector>

namespace tddp4k {

struct JitKernel {
  cudaLibrary_t lib = nullptr;
  cudaKernel_t fn = nullptr;
  int regs = 0;
};

class Jit {
 public:
  // source = prelude + kernel file; headers: (include name, text).  Returns false and fills err on any failure.
  static bool compile(const std::string &key, const std::string &source, const char *entry,
                      const std::vector<std::pair<const char *, const char *>> &headers, JitKernel *out, std::string *err) {
    static std::mutex mu;
    static std::map<std::string, JitKernel> cache;
    std::lock_guard<std::mutex> lock(mu);
    auto it = cache.find(key);
    if (it != cache.end()) { *out = it->second; return true; }
    Api &A = api();
    if (!A.ok) { *err = A.err; return false; }
    void *prog = nullptr;
    std::vector<const char *> htext, hname;
    for (auto &h : headers) { hname.push_back(h.first); htext.push_back(h.second); }
    int rc = A.create(&prog, source.c_str(), (std::string(entry) + ".cu").c_str(), (int)headers.size(), htext.data(), hname.data());
    if (rc) { *err = std::string("nvrtcCreateProgram: ") + A.errstr(rc); return false; }
    const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo"};
    rc = A.compile(prog, 3, opts);
    if (rc) {
      size_t ls = 0;
      A.logsize(prog, &ls);
      std::string log(ls, '\0');
      if (ls) A.log(prog, &log[0]);
      *err = std::string("nvrtcCompileProgram: ") + A.errstr(rc) + "\n" + log;
      A.destroy(&prog);
      return false;
    }
    size_t cs = 0;
    A.cubinsize(prog, &cs);
    std::vector<char> cubin(cs);
    rc = A.cubin(prog, cubin.data());
    A.destroy(&prog);
    if (rc || cs == 0) { *err = std::string("nvrtcGetCUBIN: ") + A.errstr(rc); return false; }
    JitKernel k;
    cudaError_t e = cudaLibraryLoadData(&k.lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e != cudaSuccess) { *err = std::string("cudaLibraryLoadData: ") + cudaGetErrorString(e); return false; }
    e = cudaLibraryGetKernel(&k.fn, k.lib, entry);
    if (e != cudaSuccess) { *err = std::string("cudaLibraryGetKernel: ") + cudaGetErrorString(e); return false; }
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, (const void *)k.fn) == cudaSuccess) k.regs = fa.numRegs;
    cache[key] = k;
    *out = k;
    return true;
  }

 private:
  struct Api {
    bool ok = false;
    std::string err;
    int (*create)(void **, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
    int (*compile)(void *, int, const char *const *) = nullptr;
    int (*cubinsize)(void *, size_t *) = nullptr;
    int (*cubin)(void *, char *) = nullptr;
    int (*logsize)(void *, size_t *) = nullptr;
    int (*log)(void *, char *) = nullptr;
    int (*destroy)(void **) = nullptr;
    const char *(*errstr)(int) = nullptr;
  };
  static Api &api() {
    static Api A = [] {
      Api a;
      const char *env = getenv("TDDP4_NVRTC");
      // the toolkit's own NVRTC first: the same compiler version as the nvcc that built the rest of the library
      const char *cands[] = {env, "/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so", "libnvrtc.so"};
      void *lib = nullptr;
      for (const char *c : cands)
        if (c && (lib = dlopen(c, RTLD_NOW | RTLD_GLOBAL))) break;
      if (!lib) { a.err = "NVRTC (libnvrtc.so.12) could not be opened; set TDDP4_NVRTC to its path"; return a; }
#define SYM(field, name)                                                              \
  *(void **)(&a.field) = dlsym(lib, name);                                           \
  if (!a.field) { a.err = std::string("NVRTC symbol missing: ") + name; return a; }
      SYM(create, "nvrtcCreateProgram") SYM(compile, "nvrtcCompileProgram") SYM(cubinsize, "nvrtcGetCUBINSize")
      SYM(cubin, "nvrtcGetCUBIN") SYM(logsize, "nvrtcGetProgramLogSize") SYM(log, "nvrtcGetProgramLog")
      SYM(destroy, "nvrtcDestroyProgram") SYM(errstr, "nvrtcGetErrorString")
#undef SYM
      a.ok = true;
      return a;
    }();
    return A;
  }
};

}  // namespace tddp4k
