// plan.cuh — host-side interpreter of the contraction plans (plans.inc): parses the plan text, owns the named
// device buffers, resolves every statement into a launch descriptor (GEMM call or permute descriptor) and enqueues
// it on the context's stream.  cclr_create executes its plan once; the sigma plan is resolved once at create time
// and replayed per trial vector with the external buffers (x1, x2, out1, out2) rebound.
#pragma once
#include "common.cuh"
#include <map>
#include <stdexcept>
#include <string>
#include <unordered_map>
#include <vector>

struct PlanError : std::runtime_error {
  int code;              // CCLR_* error code
  cudaError_t cuda;
  PlanError(int c, const std::string &m, cudaError_t e = cudaSuccess) : std::runtime_error(m), code(c), cuda(e) {}
};

struct PlanAxis { char kind, l0, l1; };   // kind: 'L' plain letter, 'P' packed pair, '1' unit
typedef std::vector<PlanAxis> PlanSpec;

enum { BUF_EXTERNAL = 0, BUF_PERSIST = 1, BUF_WORK = 2, BUF_TEMP = 3 };
enum { PHASE_OTHER = 0, PHASE_LADDER = 1, PHASE_RING = 2, PHASE_GEMM = 3, PHASE_LAYOUT = 4 };

struct PlanBuf {
  std::string name;
  PlanSpec axes;
  c128 *ptr = nullptr;
  size_t cap = 0;        // elements
  int cls = BUF_EXTERNAL;
  bool owned = false;
};

struct PlanStmt {
  std::vector<std::string> tok;
  int phase = PHASE_OTHER;
  std::vector<PlanStmt> body;   // chunk loops
};

struct ResolvedOp {
  int type = 0;                 // 0 = gemm, 1 = permute
  int phase = PHASE_OTHER;
  std::string text;             // the plan statement (profiling output)
  // gemm
  int M = 0, N = 0, K = 0, a = -1, b = -1, c = -1;
  size_t aoff = 0, boff = 0, coff = 0;
  long lda = 0, ldb = 0, ldc = 0;
  bool conjA = false, conjB = false, kn = false, acc = false;
  c128 alpha = {1.0, 0.0};
  int alpha_scalar = -1;
  // permute
  int special = 0;              // 1..5: one of the specialised layout kernels of layout.cu (see Plan::launch), 0: generic gather
  int sp_n = 0, sp_o = 0;       // their extents
  long sp_len = 0;
  PermArgs args;
  int dst = -1;
  size_t dstoff = 0;
  int srcbuf[PERM_MAX_SRC];
  int src_scalar[PERM_MAX_SRC];
};

class Plan {
 public:
  Plan(int o, int v, cudaStream_t st) : o_(o), v_(v), st_(st) {}
  ~Plan();
  Plan(const Plan &) = delete;
  Plan &operator=(const Plan &) = delete;

  void set_workspace(const ZgemmWorkspace *ws) { ws_ = ws; }
  void set_chunk_override(int len) { chunk_override_ = len; }
  void set_scalar(int id, c128 v) { scalars_[id] = v; }

  // external buffer (not owned); ptr may be null at compile time and rebound later
  void bind(const std::string &name, const std::string &spec, c128 *ptr);
  void rebind(int id, c128 *ptr) { bufs_[id].ptr = ptr; }
  // adopt an allocation made elsewhere as an owned buffer of class cls
  void adopt(const std::string &name, const std::string &spec, c128 *ptr, int cls, bool owned);
  int find(const std::string &name) const;
  const PlanBuf &buf(int id) const { return bufs_[id]; }
  size_t buf_elems(int id) const;   // current logical size

  // parse + allocate + resolve + launch, statement by statement (cclr_create)
  void execute(const char *text);
  // parse + allocate + resolve without launching (sigma plan)
  void compile(const char *text, std::vector<ResolvedOp> &ops);
  void launch(const ResolvedOp &op);

  void free_class(int cls);
  size_t owned_bytes() const { return owned_bytes_; }
  cudaStream_t stream() const { return st_; }
  void set_stream(cudaStream_t st) { st_ = st; }   // CUDA-graph capture of a compiled plan runs on a capture stream

 private:
  int o_, v_;
  cudaStream_t st_;
  const ZgemmWorkspace *ws_ = nullptr;
  int chunk_override_ = 0;
  std::vector<PlanBuf> bufs_;
  std::unordered_map<std::string, int> index_;
  std::map<char, std::pair<int, int>> chunk_;   // upper-case letter -> (offset, length)
  std::map<char, int> chunk_max_;
  c128 scalars_[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
  size_t owned_bytes_ = 0;

  static std::vector<PlanStmt> parse(const char *text);
  void run(const std::vector<PlanStmt> &stmts, std::vector<ResolvedOp> *collect);
  void declare(const PlanStmt &s);
  void release(int id);
  ResolvedOp resolve_gemm(const PlanStmt &s);
  ResolvedOp resolve_perm(const PlanStmt &s);
  void classify_special(const PlanStmt &s, ResolvedOp &r);

  int full_extent(char letter) const;
  int extent(char letter) const;
  long axis_extent(const PlanAxis &a) const;
  long axis_max_extent(const PlanAxis &a) const;
  struct View { int buf; size_t off; long rows, cols; };
  View gemm_view(const std::string &ref);
  void build_slots(int buf, const PlanSpec &access, const std::map<char, int> &ids, PermSlot *slots, int &nslot,
                   const std::string &where);
};
