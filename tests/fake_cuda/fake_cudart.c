/* fake_cudart.c -- a stand-in for the CUDA runtime, TEST INFRASTRUCTURE ONLY (tests/test_host_logic_fake_runtime.py).
 *
 * libgmco's host code (argument checks, arena carving, copies, graph construction, launch dispatch, statistics) is
 * linked against this file instead of libcudart so that it can be driven on a machine WITHOUT a GPU.  Kernels are not
 * executed: cudaLaunchKernel validates and records the launch (kernel name, grid, block, dynamic shared memory) and
 * returns.  "Device" memory is zero-filled host memory; every copy / memset is range-checked against the allocation
 * it touches and a violation is recorded.  Nothing here computes any step of the method, and the product never links it.
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef int cudaError_t;
typedef struct { unsigned x, y, z; } dim3;
typedef void* cudaStream_t;
typedef void* cudaEvent_t;
typedef void* cudaGraph_t;
typedef void* cudaGraphExec_t;
typedef void* cudaGraphNode_t;
typedef void* cudaMemPool_t;
typedef unsigned long long cudaGraphConditionalHandle;

enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2, cudaErrorInvalidConfiguration = 9 };

#define MAX_ALLOC 4096
#define MAX_FUNC 512
#define MAX_LAUNCH 65536
static struct { char* p; size_t n; } g_alloc[MAX_ALLOC];
static int g_nalloc;
static struct { const void* host; char name[160]; } g_func[MAX_FUNC];
static int g_nfunc;
typedef struct { char name[160]; unsigned gx, gy, gz, bx, by, bz; size_t smem; int captured; } launch_rec;
static launch_rec g_launch[MAX_LAUNCH];
static int g_nlaunch, g_violations, g_capturing, g_graph_launches;
static char g_violation_msg[512];
static cudaError_t g_last;
static int g_sm_count = 148;

static void violation(const char* what, const void* p, size_t n) {
  if (!g_violations) snprintf(g_violation_msg, sizeof g_violation_msg, "%s: %p + %zu", what, p, n);
  g_violations++;
}
/* the allocation that holds p, or -1 (then p is a host pointer and cannot be checked) */
static int find(const void* p) {
  for (int i = 0; i < g_nalloc; ++i)
    if (g_alloc[i].p && (const char*)p >= g_alloc[i].p && (const char*)p < g_alloc[i].p + g_alloc[i].n) return i;
  return -1;
}
static void check(const char* what, const void* p, size_t n) {
  if (!p) { if (n) violation(what, p, n); return; }
  const int i = find(p);
  if (i >= 0 && (const char*)p + n > g_alloc[i].p + g_alloc[i].n) violation(what, p, n);
}

/* ---- test hooks (read through ctypes) ---- */
int fake_violations(void) { return g_violations; }
const char* fake_violation_message(void) { return g_violation_msg; }
int fake_live_allocations(void) { int c = 0; for (int i = 0; i < g_nalloc; ++i) c += g_alloc[i].p != NULL; return c; }
int fake_launch_count(void) { return g_nlaunch; }
int fake_graph_launches(void) { return g_graph_launches; }
void fake_reset_launches(void) { g_nlaunch = 0; g_graph_launches = 0; }
void fake_set_sm_count(int n) { g_sm_count = n; }
int fake_launch(int i, char* name, int cap, unsigned* dims /* [6] */, unsigned long long* smem, int* captured) {
  if (i < 0 || i >= g_nlaunch) return -1;
  snprintf(name, (size_t)cap, "%s", g_launch[i].name);
  dims[0] = g_launch[i].gx; dims[1] = g_launch[i].gy; dims[2] = g_launch[i].gz;
  dims[3] = g_launch[i].bx; dims[4] = g_launch[i].by; dims[5] = g_launch[i].bz;
  *smem = g_launch[i].smem; *captured = g_launch[i].captured;
  return 0;
}
/* Fault injection: the library clears its 4-int device error word with the only 16-byte memset it issues.  With a
 * planted word that memset writes {code, site, block, detail} instead of zeros, as if a kernel had reported an error. */
static int g_plant[4], g_plant_on;
void fake_plant_error_word(int on, int code, int site, int block, int detail) {
  g_plant_on = on; g_plant[0] = code; g_plant[1] = site; g_plant[2] = block; g_plant[3] = detail;
}

/* ---- registration (called from nvcc's static initialisers) ---- */
void** __cudaRegisterFatBinary(void* bin) { (void)bin; static void* h; return &h; }
void __cudaRegisterFatBinaryEnd(void** h) { (void)h; }
void __cudaUnregisterFatBinary(void** h) { (void)h; }
void __cudaRegisterFunction(void** h, const char* hostFun, char* deviceFun, const char* deviceName, int tl, void* tid,
                            void* bid, void* bdim, void* gdim, int* wsize) {
  (void)h; (void)deviceFun; (void)tl; (void)tid; (void)bid; (void)bdim; (void)gdim; (void)wsize;
  if (g_nfunc < MAX_FUNC) { g_func[g_nfunc].host = hostFun; snprintf(g_func[g_nfunc].name, 160, "%s", deviceName); g_nfunc++; }
}
static dim3 g_cfg_grid, g_cfg_block; static size_t g_cfg_smem; static cudaStream_t g_cfg_stream;
unsigned __cudaPushCallConfiguration(dim3 grid, dim3 block, size_t smem, cudaStream_t st) {
  g_cfg_grid = grid; g_cfg_block = block; g_cfg_smem = smem; g_cfg_stream = st; return 0;
}
cudaError_t __cudaPopCallConfiguration(dim3* grid, dim3* block, size_t* smem, void* st) {
  *grid = g_cfg_grid; *block = g_cfg_block; *smem = g_cfg_smem; *(cudaStream_t*)st = g_cfg_stream; return cudaSuccess;
}

static size_t g_func_smem_cap[MAX_FUNC];
static int func_index(const void* f) { for (int i = 0; i < g_nfunc; ++i) if (g_func[i].host == f) return i; return -1; }

cudaError_t cudaLaunchKernel(const void* func, dim3 grid, dim3 block, void** args, size_t smem, cudaStream_t st) {
  (void)args; (void)st;
  const int fi = func_index(func);
  const size_t cap = fi >= 0 && g_func_smem_cap[fi] ? g_func_smem_cap[fi] : 48 * 1024;
  if (!grid.x || !grid.y || !grid.z || !block.x || !block.y || !block.z || block.x * block.y * block.z > 1024 ||
      grid.y > 65535 || grid.z > 65535 || smem > cap) {
    g_last = cudaErrorInvalidConfiguration; return g_last;
  }
  if (g_nlaunch < MAX_LAUNCH) {
    launch_rec* r = &g_launch[g_nlaunch++];
    snprintf(r->name, 160, "%s", fi >= 0 ? g_func[fi].name : "?");
    r->gx = grid.x; r->gy = grid.y; r->gz = grid.z; r->bx = block.x; r->by = block.y; r->bz = block.z; r->smem = smem;
    r->captured = g_capturing;
  }
  return cudaSuccess;
}
cudaError_t cudaFuncSetAttribute(const void* func, int attr, int value) {
  const int fi = func_index(func);
  if (fi < 0 || attr != 8 /* cudaFuncAttributeMaxDynamicSharedMemorySize */ || value < 0 || value > 227 * 1024) return cudaErrorInvalidValue;
  g_func_smem_cap[fi] = (size_t)value;
  return cudaSuccess;
}

/* ---- device, errors ---- */
cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int* v, int attr, int dev) {
  (void)dev;
  if (attr == 75) *v = 10;            /* cudaDevAttrComputeCapabilityMajor */
  else if (attr == 16) *v = g_sm_count;   /* cudaDevAttrMultiProcessorCount */
  else *v = 0;
  return cudaSuccess;
}
cudaError_t cudaGetLastError(void) { cudaError_t e = g_last; g_last = cudaSuccess; return e; }
cudaError_t cudaPeekAtLastError(void) { return g_last; }
const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : e == 9 ? "invalid configuration argument" : "fake runtime error"; }
cudaError_t cudaDeviceGetDefaultMemPool(cudaMemPool_t* p, int dev) { (void)dev; static int pool; *p = &pool; return cudaSuccess; }
cudaError_t cudaMemPoolSetAttribute(cudaMemPool_t p, int a, void* v) { (void)p; (void)a; (void)v; return cudaSuccess; }

/* ---- memory ---- */
cudaError_t cudaMallocAsync(void** p, size_t n, cudaStream_t st) {
  (void)st;
  int slot = -1;
  for (int i = 0; i < g_nalloc; ++i) if (!g_alloc[i].p) { slot = i; break; }
  if (slot < 0) { if (g_nalloc >= MAX_ALLOC) return cudaErrorMemoryAllocation; slot = g_nalloc++; }
  char* q = (char*)calloc(n ? n : 1, 1);
  if (!q) return cudaErrorMemoryAllocation;
  g_alloc[slot].p = q; g_alloc[slot].n = n; *p = q;
  return cudaSuccess;
}
cudaError_t cudaFreeAsync(void* p, cudaStream_t st) {
  (void)st;
  for (int i = 0; i < g_nalloc; ++i) if (g_alloc[i].p == p) { free(p); g_alloc[i].p = NULL; return cudaSuccess; }
  violation("cudaFreeAsync of a pointer that is not a live allocation", p, 0);
  return cudaErrorInvalidValue;
}
struct cudaPointerAttributes { int type; int device; void* devicePointer; void* hostPointer; };
cudaError_t cudaPointerGetAttributes(struct cudaPointerAttributes* a, const void* p) {
  memset(a, 0, sizeof *a);
  a->type = find(p) >= 0 ? 2 /* cudaMemoryTypeDevice */ : 0 /* unregistered host */;
  return cudaSuccess;
}
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, int kind, cudaStream_t st) {
  (void)kind; (void)st;
  check("cudaMemcpy destination", d, n); check("cudaMemcpy source", s, n);
  if (d && s && n) memmove(d, s, n);
  return cudaSuccess;
}
cudaError_t cudaMemcpy(void* d, const void* s, size_t n, int kind) { return cudaMemcpyAsync(d, s, n, kind, NULL); }
cudaError_t cudaMemcpy2DAsync(void* d, size_t dp, const void* s, size_t sp, size_t w, size_t h, int kind, cudaStream_t st) {
  (void)kind; (void)st;
  if (w > dp || w > sp) { violation("cudaMemcpy2D width above pitch", d, w); return cudaErrorInvalidValue; }
  if (h) { check("cudaMemcpy2D destination", d, (h - 1) * dp + w); check("cudaMemcpy2D source", s, (h - 1) * sp + w); }
  for (size_t r = 0; r < h; ++r) memmove((char*)d + r * dp, (const char*)s + r * sp, w);
  return cudaSuccess;
}
cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t st) {
  (void)st;
  if (find(d) < 0) violation("cudaMemset of a pointer that is not device memory", d, n);
  check("cudaMemset", d, n);
  if (find(d) >= 0) memset(d, v, n);
  if (g_plant_on && n == 16 && find(d) >= 0) memcpy(d, g_plant, 16);
  return cudaSuccess;
}

/* ---- streams, events ---- */
cudaError_t cudaStreamSynchronize(cudaStream_t st) { (void)st; return cudaSuccess; }
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* st, unsigned f) { (void)f; *st = malloc(8); return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t st) { free(st); return cudaSuccess; }
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = malloc(8); return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t e) { free(e); return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t st) { (void)st; return e ? cudaSuccess : cudaErrorInvalidValue; }
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) { if (!a || !b) return cudaErrorInvalidValue; *ms = 0.01f; return cudaSuccess; }

/* ---- graphs: constructed, never executed ---- */
struct fakeGraphNodeParams {                  /* prefix of cudaGraphNodeParams that the library touches */
  int type; int reserved0[3];
  struct { cudaGraphConditionalHandle handle; int type; unsigned size; cudaGraph_t* phGraph_out; } conditional;
};
cudaError_t cudaGraphCreate(cudaGraph_t* g, unsigned f) { (void)f; *g = calloc(1, 64); return cudaSuccess; }
cudaError_t cudaGraphDestroy(cudaGraph_t g) { free(g); return cudaSuccess; }
cudaError_t cudaGraphConditionalHandleCreate(cudaGraphConditionalHandle* h, cudaGraph_t g, unsigned dflt, unsigned flags) {
  (void)g; (void)dflt; (void)flags; *h = 0x1234; return cudaSuccess;
}
cudaError_t cudaGraphAddNode(cudaGraphNode_t* node, cudaGraph_t g, const cudaGraphNode_t* deps, size_t ndeps, void* params) {
  (void)g; (void)deps; (void)ndeps;
  struct fakeGraphNodeParams* p = (struct fakeGraphNodeParams*)params;
  if (p->type != 13 /* cudaGraphNodeTypeConditional */ || p->conditional.size != 1) return cudaErrorInvalidValue;
  static cudaGraph_t body[1];
  body[0] = calloc(1, 64);                    /* leaked on purpose: owned by the parent graph in the real runtime */
  p->conditional.phGraph_out = body;
  *node = body;
  return cudaSuccess;
}
cudaError_t cudaStreamBeginCaptureToGraph(cudaStream_t st, cudaGraph_t g, const cudaGraphNode_t* deps, const void* dd, size_t nd, int mode) {
  (void)st; (void)deps; (void)dd; (void)nd; (void)mode;
  if (!g || g_capturing) return cudaErrorInvalidValue;
  g_capturing = 1; return cudaSuccess;
}
cudaError_t cudaStreamEndCapture(cudaStream_t st, cudaGraph_t* g) { (void)st; if (g) *g = NULL; if (!g_capturing) return cudaErrorInvalidValue; g_capturing = 0; return cudaSuccess; }
cudaError_t cudaGraphInstantiate(cudaGraphExec_t* e, cudaGraph_t g, unsigned long long f) { (void)f; if (!g) return cudaErrorInvalidValue; *e = malloc(8); return cudaSuccess; }
cudaError_t cudaGraphExecDestroy(cudaGraphExec_t e) { free(e); return cudaSuccess; }
cudaError_t cudaGraphLaunch(cudaGraphExec_t e, cudaStream_t st) { (void)st; if (!e) return cudaErrorInvalidValue; g_graph_launches++; return cudaSuccess; }

/* ---- driver entry point: a cuTensorMapEncodeTiled that checks what the real one checks ---- */
static int g_tensor_maps;
int fake_tensor_maps(void) { return g_tensor_maps; }
static int fake_cuTensorMapEncodeTiled(void* map, int dtype, unsigned rank, void* addr, const uint64_t* dims, const uint64_t* strides,
                                       const uint32_t* box, const uint32_t* estr, int interleave, int swizzle, int l2, int oob) {
  (void)interleave; (void)l2; (void)oob;
  if (!map || !addr || rank < 1 || rank > 5 || ((uintptr_t)addr & 15) || dtype != 7 /* FLOAT32 */) return 1;
  if (find(addr) < 0) { violation("tensor map over memory that is not a device allocation", addr, 0); return 1; }
  uint64_t extent = 4;
  for (unsigned i = 0; i < rank; ++i) {
    if (!dims[i] || dims[i] > (1ull << 32) || !box[i] || box[i] > 256 || estr[i] != 1) return 1;
    if (i + 1 < rank && ((strides[i] & 15) || strides[i] >= (1ull << 40))) return 1;
  }
  const uint64_t inner = (uint64_t)box[0] * 4;
  if (swizzle == 3 /* 128B */ || swizzle == 4 /* 128B_ATOM_32B */) { if (inner > 128) return 1; }
  else if (swizzle != 0) return 1;
  /* the whole tensor must lie inside the allocation: last element of the last row */
  extent = dims[0] * 4;
  for (unsigned i = 1; i < rank; ++i) { const uint64_t e = (dims[i] - 1) * strides[i - 1] + dims[0] * 4; if (e > extent) extent = e; }
  {
    uint64_t far = dims[0] * 4;
    for (unsigned i = 1; i < rank; ++i) far += (dims[i] - 1) * strides[i - 1];
    check("tensor map extent", addr, (size_t)far);
  }
  memset(map, 0, 128);
  g_tensor_maps++;
  return 0;
}
cudaError_t cudaGetDriverEntryPoint(const char* name, void** fn, unsigned long long flags, int* status) {
  (void)flags;
  if (strcmp(name, "cuTensorMapEncodeTiled")) { *fn = NULL; if (status) *status = 1; return cudaErrorInvalidValue; }
  *fn = (void*)fake_cuTensorMapEncodeTiled; if (status) *status = 0; return cudaSuccess;
}
