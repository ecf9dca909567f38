// plan.cu — parser and executor of the contraction plans (see plan.cuh, plans.inc).
#include "plan.cuh"
#include "../../include/cclr.h"
#include <cctype>
#include <cstdlib>
#include <sstream>

namespace {

bool is_occ(char l) {
  l = (char)std::tolower((unsigned char)l);
  return l >= 'i' && l <= 'n';
}
bool is_vir(char l) {
  l = (char)std::tolower((unsigned char)l);
  return l >= 'a' && l <= 'h';
}

// "(ab)E;j" -> groups of axes
std::vector<PlanSpec> parse_spec(const std::string &s) {
  std::vector<PlanSpec> groups(1);
  for (size_t k = 0; k < s.size();) {
    const char c = s[k];
    if (c == ';') {
      groups.emplace_back();
      ++k;
    } else if (c == '(') {
      if (k + 3 >= s.size() || s[k + 3] != ')') throw PlanError(CCLR_EINVAL, "bad pair in spec " + s);
      groups.back().push_back(PlanAxis{'P', s[k + 1], s[k + 2]});
      k += 4;
    } else if (c == '1') {
      groups.back().push_back(PlanAxis{'1', 0, 0});
      ++k;
    } else if (is_occ(c) || is_vir(c)) {
      groups.back().push_back(PlanAxis{'L', c, 0});
      ++k;
    } else {
      throw PlanError(CCLR_EINVAL, "bad character in spec " + s);
    }
  }
  return groups;
}

PlanSpec flat_spec(const std::string &s) {
  PlanSpec out;
  for (auto &g : parse_spec(s)) out.insert(out.end(), g.begin(), g.end());
  return out;
}

// "name[spec]" -> (name, spec)
void split_ref(const std::string &tok, std::string &name, std::string &spec) {
  const size_t lb = tok.find('['), rb = tok.rfind(']');
  if (lb == std::string::npos || rb == std::string::npos || rb < lb) throw PlanError(CCLR_EINVAL, "bad reference " + tok);
  name = tok.substr(0, lb);
  spec = tok.substr(lb + 1, rb - lb - 1);
}

void cuda_check(cudaError_t e, const std::string &where) {
  if (e != cudaSuccess)
    throw PlanError(e == cudaErrorMemoryAllocation ? CCLR_ENOMEM : CCLR_ECUDA,
                    where + ": " + cudaGetErrorString(e), e);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
Plan::~Plan() {
  for (auto &b : bufs_)
    if (b.owned && b.ptr) cudaFree(b.ptr);
}

int Plan::full_extent(char letter) const {
  if (is_occ(letter)) return o_;
  if (is_vir(letter)) return v_;
  throw PlanError(CCLR_EINVAL, std::string("unknown index letter ") + letter);
}

int Plan::extent(char letter) const {
  if (std::isupper((unsigned char)letter)) {
    auto it = chunk_.find(letter);
    if (it == chunk_.end()) throw PlanError(CCLR_EINVAL, std::string("chunk letter outside its loop: ") + letter);
    return it->second.second;
  }
  return full_extent(letter);
}

long Plan::axis_extent(const PlanAxis &a) const {
  if (a.kind == '1') return 1;
  if (a.kind == 'L') return extent(a.l0);
  return npair(full_extent(a.l0));
}

long Plan::axis_max_extent(const PlanAxis &a) const {
  if (a.kind == 'L' && std::isupper((unsigned char)a.l0)) {
    auto it = chunk_max_.find(a.l0);
    if (it == chunk_max_.end()) throw PlanError(CCLR_EINVAL, "chunk letter without a loop");
    return it->second;
  }
  return axis_extent(a);
}

int Plan::find(const std::string &name) const {
  auto it = index_.find(name);
  return it == index_.end() ? -1 : it->second;
}

size_t Plan::buf_elems(int id) const {
  size_t n = 1;
  for (auto &a : bufs_[id].axes) n *= (size_t)axis_extent(a);
  return n;
}

void Plan::bind(const std::string &name, const std::string &spec, c128 *ptr) {
  adopt(name, spec, ptr, BUF_EXTERNAL, false);
}

void Plan::adopt(const std::string &name, const std::string &spec, c128 *ptr, int cls, bool owned) {
  int id = find(name);
  if (id < 0) {
    id = (int)bufs_.size();
    bufs_.emplace_back();
    index_[name] = id;
  } else if (bufs_[id].owned && bufs_[id].ptr) {
    throw PlanError(CCLR_EINVAL, "rebinding an owned buffer " + name);
  }
  PlanBuf &b = bufs_[id];
  b.name = name;
  b.axes = flat_spec(spec);
  b.ptr = ptr;
  b.cls = cls;
  b.owned = owned;
  b.cap = 1;
  for (auto &a : b.axes) b.cap *= (size_t)axis_max_extent(a);
  if (owned) owned_bytes_ += b.cap * sizeof(c128);
}

void Plan::declare(const PlanStmt &s) {
  if (s.tok.size() < 4) throw PlanError(CCLR_EINVAL, "buf needs name, spec, class");
  const std::string &name = s.tok[1];
  const int id = find(name);
  if (id >= 0 && bufs_[id].ptr) return;   // already allocated (chunk loop iteration > 0, or sigma recompiled)
  const int cls = s.tok[3] == "persist" ? BUF_PERSIST : s.tok[3] == "work" ? BUF_WORK : BUF_TEMP;
  PlanSpec axes = flat_spec(s.tok[2]);
  size_t cap = 1;
  for (auto &a : axes) cap *= (size_t)axis_max_extent(a);
  c128 *ptr = nullptr;
  cuda_check(cudaMalloc(&ptr, (cap ? cap : 1) * sizeof(c128)), "cudaMalloc(" + name + ")");
  adopt(name, s.tok[2], ptr, cls, true);
}

void Plan::release(int id) {
  PlanBuf &b = bufs_[id];
  if (b.owned && b.ptr) {
    cuda_check(cudaStreamSynchronize(st_), "sync before free");
    cuda_check(cudaFree(b.ptr), "cudaFree(" + b.name + ")");
    owned_bytes_ -= b.cap * sizeof(c128);
  }
  b.ptr = nullptr;
  b.owned = false;
}

void Plan::free_class(int cls) {
  for (size_t i = 0; i < bufs_.size(); ++i)
    if (bufs_[i].cls == cls && bufs_[i].owned) release((int)i);
}

// ---------------------------------------------------------------------------------------------------------------
std::vector<PlanStmt> Plan::parse(const char *text) {
  std::vector<PlanStmt> top;
  std::vector<std::vector<PlanStmt> *> stack{&top};
  std::istringstream in(text);
  std::string line;
  int phase = PHASE_OTHER;
  while (std::getline(in, line)) {
    const size_t hash = line.find('#');
    if (hash != std::string::npos) line.resize(hash);
    std::istringstream ls(line);
    PlanStmt s;
    std::string t;
    while (ls >> t) s.tok.push_back(t);
    if (s.tok.empty()) continue;
    const std::string &op = s.tok[0];
    if (op[0] == '@') {
      phase = op == "@ladder" ? PHASE_LADDER : op == "@ring" ? PHASE_RING : op == "@gemm" ? PHASE_GEMM
              : op == "@layout" ? PHASE_LAYOUT : PHASE_OTHER;
      continue;
    }
    s.phase = phase;
    if (op == "end") {
      if (stack.size() < 2) throw PlanError(CCLR_EINVAL, "end without chunk");
      stack.pop_back();
      continue;
    }
    stack.back()->push_back(s);
    if (op == "chunk") stack.push_back(&stack.back()->back().body);
  }
  if (stack.size() != 1) throw PlanError(CCLR_EINVAL, "chunk without end");
  return top;
}

void Plan::execute(const char *text) { run(parse(text), nullptr); }

void Plan::compile(const char *text, std::vector<ResolvedOp> &ops) { run(parse(text), &ops); }

void Plan::run(const std::vector<PlanStmt> &stmts, std::vector<ResolvedOp> *collect) {
  for (const PlanStmt &s : stmts) {
    const std::string &op = s.tok[0];
    if (op == "buf") {
      declare(s);
    } else if (op == "free") {
      const int id = find(s.tok.at(1));
      if (id < 0) throw PlanError(CCLR_EINVAL, "free of unknown buffer " + s.tok[1]);
      release(id);
    } else if (op == "chunk") {
      if (collect) throw PlanError(CCLR_EINVAL, "chunk loops are not allowed in a compiled plan");
      const char letter = s.tok.at(1)[0];
      int len = std::atoi(s.tok.at(2).c_str());
      if (chunk_override_ > 0) len = chunk_override_;
      const int full = full_extent(letter);
      if (len > full) len = full;
      if (len < 1) len = 1;
      chunk_max_[letter] = len;
      std::vector<int> created;
      for (int off = 0; off < full; off += len) {
        chunk_[letter] = std::make_pair(off, std::min(len, full - off));
        const size_t before = bufs_.size();
        run(s.body, nullptr);
        for (size_t i = before; i < bufs_.size(); ++i) created.push_back((int)i);
      }
      // buffers declared inside the loop die with it
      for (const PlanStmt &b : s.body)
        if (b.tok[0] == "buf") {
          const int id = find(b.tok[1]);
          if (id >= 0) release(id);
        }
      chunk_.erase(letter);
      chunk_max_.erase(letter);
    } else if (op == "gemm" || op == "perm" || op == "scat") {
      ResolvedOp r = op == "gemm" ? resolve_gemm(s) : resolve_perm(s);
      r.phase = s.phase;
      for (auto &t : s.tok) r.text += (r.text.empty() ? "" : " ") + t;
      if (collect)
        collect->push_back(r);
      else
        launch(r);
    } else {
      throw PlanError(CCLR_EINVAL, "unknown plan statement " + op);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
Plan::View Plan::gemm_view(const std::string &ref) {
  std::string name, spec;
  split_ref(ref, name, spec);
  const int id = find(name);
  if (id < 0) throw PlanError(CCLR_EINVAL, "gemm: unknown buffer " + name);
  std::vector<PlanSpec> groups = parse_spec(spec);
  if (groups.size() != 2) throw PlanError(CCLR_EINVAL, "gemm operand needs rows;cols: " + ref);
  PlanSpec acc, decl;
  for (auto &g : groups)
    for (auto &a : g)
      if (a.kind != '1') acc.push_back(a);
  for (auto &a : bufs_[id].axes)
    if (a.kind != '1') decl.push_back(a);
  if (acc.size() != decl.size()) throw PlanError(CCLR_EINVAL, "gemm view rank mismatch " + ref);
  size_t base = 0;
  for (size_t k = 0; k < acc.size(); ++k) {
    const PlanAxis &d = decl[k], &a = acc[k];
    bool ok = false;
    if (d.kind == 'L' && a.kind == 'L' && full_extent(d.l0) == full_extent(a.l0)) {
      const bool du = std::isupper((unsigned char)d.l0), au = std::isupper((unsigned char)a.l0);
      if (d.l0 == a.l0) {
        ok = true;
      } else if (k == 0 && au && !du) {
        size_t rest = 1;
        for (size_t j = 1; j < decl.size(); ++j) rest *= (size_t)axis_extent(decl[j]);
        base = (size_t)chunk_.at(a.l0).first * rest;
        ok = true;
      } else if (!du && !au) {
        ok = true;   // renamed letter of the same range
      }
    } else if (d.kind == 'P' && a.kind == 'P' && full_extent(d.l0) == full_extent(a.l0)) {
      ok = true;
    }
    if (!ok) throw PlanError(CCLR_EINVAL, "gemm view does not match the declared layout: " + ref);
  }
  View v;
  v.buf = id;
  v.off = base;
  v.rows = 1;
  v.cols = 1;
  for (auto &a : groups[0]) v.rows *= axis_extent(a);
  for (auto &a : groups[1]) v.cols *= axis_extent(a);
  if (base + (size_t)v.rows * (size_t)v.cols > bufs_[id].cap) throw PlanError(CCLR_EINVAL, "gemm view exceeds buffer " + ref);
  return v;
}

ResolvedOp Plan::resolve_gemm(const PlanStmt &s) {
  // gemm C[rows;cols] (=|+=) alpha [conj] A[..] [conj] B[..] nk|kn
  ResolvedOp r;
  r.type = 0;
  size_t k = 1;
  const View C = gemm_view(s.tok.at(k++));
  const std::string acc = s.tok.at(k++);
  r.acc = acc == "+=";
  if (!r.acc && acc != "=") throw PlanError(CCLR_EINVAL, "gemm needs = or +=");
  const std::string al = s.tok.at(k++);
  if (al[0] == '$') {
    r.alpha_scalar = 0;
  } else {
    r.alpha = make_double2(std::atof(al.c_str()), 0.0);
  }
  if (s.tok.at(k) == "conj") { r.conjA = true; ++k; }
  const View A = gemm_view(s.tok.at(k++));
  if (s.tok.at(k) == "conj") { r.conjB = true; ++k; }
  const View B = gemm_view(s.tok.at(k++));
  const std::string mode = s.tok.at(k++);
  r.kn = mode == "kn";
  if (!r.kn && mode != "nk") throw PlanError(CCLR_EINVAL, "gemm needs nk or kn");
  r.M = (int)C.rows;
  r.N = (int)C.cols;
  r.K = (int)A.cols;
  const long bk = r.kn ? B.rows : B.cols, bn = r.kn ? B.cols : B.rows;
  if (A.rows != C.rows || bk != A.cols || bn != C.cols) {
    std::string line;
    for (auto &t : s.tok) line += t + " ";
    throw PlanError(CCLR_EINVAL, "gemm shape mismatch: " + line);
  }
  r.a = A.buf; r.b = B.buf; r.c = C.buf;
  r.aoff = A.off; r.boff = B.off; r.coff = C.off;
  r.lda = A.cols; r.ldb = B.cols; r.ldc = C.cols;
  return r;
}

void Plan::build_slots(int buf, const PlanSpec &access, const std::map<char, int> &ids, PermSlot *slots, int &nslot,
                       const std::string &where) {
  const PlanSpec &decl = bufs_[buf].axes;
  if (decl.size() != access.size() || decl.size() > (size_t)PERM_MAX_SLOTS)
    throw PlanError(CCLR_EINVAL, "perm: rank mismatch for " + where);
  std::vector<long> stride(decl.size(), 1);
  for (int k = (int)decl.size() - 2; k >= 0; --k) stride[k] = stride[k + 1] * axis_extent(decl[k + 1]);
  nslot = (int)decl.size();
  for (size_t k = 0; k < decl.size(); ++k) {
    const PlanAxis &d = decl[k], &a = access[k];
    PermSlot &sl = slots[k];
    sl.stride = stride[k];
    sl.sub = 0;
    sl.l0 = sl.l1 = 0;
    if (d.kind == '1') {
      if (a.kind != '1') throw PlanError(CCLR_EINVAL, "perm: unit axis mismatch in " + where);
      sl.kind = 2;
    } else if (d.kind == 'L') {
      if (a.kind != 'L' || full_extent(d.l0) != full_extent(a.l0) || !ids.count(a.l0))
        throw PlanError(CCLR_EINVAL, "perm: plain axis mismatch in " + where);
      sl.kind = 0;
      sl.l0 = ids.at(a.l0);
      if (std::isupper((unsigned char)d.l0)) sl.sub = chunk_.at(d.l0).first;
    } else {
      if (a.kind != 'P' || full_extent(d.l0) != full_extent(a.l0) || full_extent(a.l0) != full_extent(a.l1) ||
          !ids.count(a.l0) || !ids.count(a.l1))
        throw PlanError(CCLR_EINVAL, "perm: pair axis mismatch in " + where);
      sl.kind = 1;
      sl.l0 = ids.at(a.l0);
      sl.l1 = ids.at(a.l1);
    }
  }
}

ResolvedOp Plan::resolve_perm(const PlanStmt &s) {
  // perm D[spec] (=|+=) c [conj] S[spec] ...            scat D[spec] += c [conj] S[spec] iter SPEC cond lt|gt|all
  ResolvedOp r;
  r.type = 1;
  PermArgs &p = r.args;
  p = PermArgs{};
  const bool scat = s.tok[0] == "scat";
  std::string line;
  for (auto &t : s.tok) line += t + " ";
  std::string dname, dspec;
  split_ref(s.tok.at(1), dname, dspec);
  r.dst = find(dname);
  if (r.dst < 0) throw PlanError(CCLR_EINVAL, "perm: unknown buffer " + dname);
  p.accumulate = s.tok.at(2) == "+=";
  if (!p.accumulate && s.tok[2] != "=") throw PlanError(CCLR_EINVAL, "perm needs = or +=");
  size_t end = s.tok.size();
  PlanSpec iter = flat_spec(dspec);
  p.cond = 0;
  if (scat) {
    size_t ii = 0;
    for (size_t k = 3; k < s.tok.size(); ++k)
      if (s.tok[k] == "iter") ii = k;
    if (!ii || ii + 3 >= s.tok.size() || s.tok[ii + 2] != "cond") throw PlanError(CCLR_EINVAL, "scat needs iter SPEC cond X: " + line);
    iter = flat_spec(s.tok[ii + 1]);
    const std::string &c = s.tok[ii + 3];
    p.cond = c == "lt" ? 1 : c == "gt" ? 2 : 0;
    end = ii;
    if (!p.accumulate) throw PlanError(CCLR_EINVAL, "scat must accumulate");
  }
  // iteration axes and letter ids
  if (iter.size() > (size_t)PERM_MAX_AXES) throw PlanError(CCLR_EINVAL, "perm: too many axes: " + line);
  std::map<char, int> ids;
  auto new_id = [&](char l) {
    if (ids.count(l)) throw PlanError(CCLR_EINVAL, "perm: letter used twice in the iteration space: " + line);
    const int id = (int)ids.size();
    if (id >= PERM_MAX_LETTERS) throw PlanError(CCLR_EINVAL, "perm: too many letters");
    ids[l] = id;
    return id;
  };
  p.naxis = (int)iter.size();
  p.total = 1;
  for (size_t k = 0; k < iter.size(); ++k) {
    PermAxis &ax = p.axis[k];
    const PlanAxis &a = iter[k];
    ax.ext = (int)axis_extent(a);
    ax.off = 0;
    ax.l0 = ax.l1 = 0;
    if (a.kind == '1') {
      ax.kind = 2;
    } else if (a.kind == 'L') {
      ax.kind = 0;
      ax.l0 = new_id(a.l0);
      if (std::isupper((unsigned char)a.l0)) ax.off = chunk_.at(a.l0).first;
    } else {
      ax.kind = 1;
      ax.l0 = new_id(a.l0);
      ax.l1 = new_id(a.l1);
    }
    p.total *= ax.ext;
  }
  // destination
  const PlanSpec dacc = flat_spec(dspec);
  build_slots(r.dst, dacc, ids, p.dslot, p.ndslot, line);
  p.dst_linear = scat ? 0 : 1;
  r.dstoff = 0;
  if (!scat) {
    // gather: the iteration space is the destination view; its origin is the offset of the first element
    for (int k = 0; k < p.ndslot; ++k) {
      const PermSlot &sl = p.dslot[k];
      if (sl.kind == 0) {
        int first = 0;
        for (int a = 0; a < p.naxis; ++a)
          if (p.axis[a].kind == 0 && p.axis[a].l0 == sl.l0) first = p.axis[a].off;
        r.dstoff += (size_t)(first - sl.sub) * (size_t)sl.stride;
      }
    }
    // the destination view must be a dense prefix: same axis kinds and extents in the same order
    const PlanSpec &decl = bufs_[r.dst].axes;
    for (size_t k = 0; k < decl.size(); ++k) {
      const bool same = decl[k].kind == dacc[k].kind &&
                        (k == 0 || decl[k].kind != 'L' || axis_extent(decl[k]) == axis_extent(dacc[k])) &&
                        (decl[k].kind != 'P' || (ids.at(dacc[k].l0) < ids.at(dacc[k].l1)));
      if (!same) throw PlanError(CCLR_EINVAL, "perm: destination is not a dense view: " + line);
    }
  } else if (p.cond) {
    bool found = false;
    for (int k = 0; k < p.ndslot && !found; ++k)
      if (p.dslot[k].kind == 1) {
        p.cond_l0 = p.dslot[k].l0;
        p.cond_l1 = p.dslot[k].l1;
        found = true;
      }
    if (!found) throw PlanError(CCLR_EINVAL, "scat cond needs a destination pair: " + line);
  }
  // sources
  p.nsrc = 0;
  for (size_t k = 3; k < end;) {
    if (p.nsrc >= PERM_MAX_SRC) throw PlanError(CCLR_EINVAL, "perm: too many sources: " + line);
    PermOperand &src = p.src[p.nsrc];
    const std::string &ct = s.tok.at(k++);
    r.src_scalar[p.nsrc] = -1;
    if (ct[0] == '$') {
      r.src_scalar[p.nsrc] = 0;
      src.coef = make_double2(0.0, 0.0);
    } else {
      src.coef = make_double2(std::atof(ct.c_str()), 0.0);
    }
    src.conj = 0;
    if (s.tok.at(k) == "conj") { src.conj = 1; ++k; }
    std::string sname, sspec;
    split_ref(s.tok.at(k++), sname, sspec);
    const int sb = find(sname);
    if (sb < 0) throw PlanError(CCLR_EINVAL, "perm: unknown buffer " + sname);
    r.srcbuf[p.nsrc] = sb;
    build_slots(sb, flat_spec(sspec), ids, src.slot, src.nslot, line);
    ++p.nsrc;
  }
  if (p.nsrc == 0) throw PlanError(CCLR_EINVAL, "perm without sources: " + line);
  classify_special(s, r);
  return r;
}

// Recognise the hot layout statements of sigma (layout.cu) by the SHAPE of their index specs: letters are renamed A, B, C, ... in
// order of first appearance in the destination spec, so "Ur[ea(ij)] = 1 x2[(ea)(ij)]" and the same statement in other letters
// of the same ranges match alike.  Anything else keeps special = 0 (generic gather kernel).
void Plan::classify_special(const PlanStmt &s, ResolvedOp &r) {
  r.special = 0;
  if (s.tok[0] != "perm") return;
  std::string dname, dspec;
  split_ref(s.tok[1], dname, dspec);
  for (char c : dspec)
    if (std::isupper((unsigned char)c) || c == '1') return;
  // the final antisymmetrised pack of sigma2, matched literally
  static const char *const FINAL[] = {"+=", "$nz", "x2[(ab)(ij)]", "1", "Y[ab(ij)]", "-1", "Y[ba(ij)]", "1", "Q[(ab)ij]", "-1", "Q[(ab)ji]",
                                      "1", "Z[bjai]", "-1", "Z[ajbi]", "-1", "Z[biaj]", "1", "Z[aibj]"};
  if (s.tok.size() == 2 + sizeof(FINAL) / sizeof(FINAL[0]) && dspec == "(ab)(ij)") {
    bool same = true;
    for (size_t k = 0; k < sizeof(FINAL) / sizeof(FINAL[0]); ++k) same = same && s.tok[2 + k] == FINAL[k];
    const size_t smem = (size_t)3 * o_ * o_ * sizeof(c128);
    if (same && smem <= LAYOUT_MAX_SMEM) { r.special = 5; r.sp_n = v_; r.sp_o = o_; }
    return;
  }
  if (s.tok.size() != 5 || s.tok[2] != "=" || s.tok[3] != "1") return;
  std::string sname, sspec;
  split_ref(s.tok[4], sname, sspec);
  std::map<char, char> ren;
  auto canon = [&](const std::string &spec, bool define) {
    std::string out;
    for (char c : spec) {
      if (c == '(' || c == ')') { out += c; continue; }
      if (!ren.count(c)) {
        if (!define) return std::string("?");
        ren[c] = (char)('A' + ren.size());
      }
      out += ren[c];
    }
    return out;
  };
  const std::string d = canon(dspec, true), q = canon(sspec, false);
  auto letter = [&](char canon_letter) {
    for (auto &kv : ren)
      if (kv.second == canon_letter) return kv.first;
    return 'a';
  };
  if (ren.size() != 4) return;
  const int eA = full_extent(letter('A')), eB = full_extent(letter('B')), eC = full_extent(letter('C')), eD = full_extent(letter('D'));
  if (d == "AB(CD)" && q == "(AB)(CD)" && eA == eB && eC == eD) {
    r.special = 1; r.sp_n = eA; r.sp_len = npair(eC);
  } else if (d == "(AB)CD" && q == "(AB)(CD)" && eA == eB && eC == eD && (size_t)npair(eC) * sizeof(c128) <= 48 * 1024) {
    r.special = 2; r.sp_len = npair(eA); r.sp_o = eC;
  } else if (d == "ABCD" && q == "(AC)(BD)" && eA == eC && eB == eD && (size_t)npair(eB) * sizeof(c128) <= 48 * 1024) {
    r.special = 3; r.sp_n = eA; r.sp_o = eB;
  } else if (d == "AB(CD)" && q == "(CD)(AB)" && eA == eB && eC == eD) {
    r.special = 4; r.sp_len = npair(eC); r.sp_o = eA;
  }
}

// ---------------------------------------------------------------------------------------------------------------
void Plan::launch(const ResolvedOp &op) {
  if (op.type == 0) {
    const PlanBuf &A = bufs_[op.a], &B = bufs_[op.b], &C = bufs_[op.c];
    if (!A.ptr || !B.ptr || !C.ptr) throw PlanError(CCLR_EINVAL, "gemm on an unbound buffer (" + A.name + "," + B.name + "," + C.name + ")");
    const c128 alpha = op.alpha_scalar >= 0 ? scalars_[op.alpha_scalar] : op.alpha;
    const c128 beta = op.acc ? make_double2(1.0, 0.0) : make_double2(0.0, 0.0);
    cuda_check(zgemm(st_, op.M, op.N, op.K, alpha, A.ptr + op.aoff, op.lda, op.conjA, B.ptr + op.boff, op.ldb, op.kn,
                     op.conjB, beta, C.ptr + op.coff, op.ldc, 1, 0, 0, 0, ws_),
               "zgemm(" + C.name + ")");
  } else if (op.special) {
    const PlanBuf &D = bufs_[op.dst];
    if (!D.ptr) throw PlanError(CCLR_EINVAL, "perm on an unbound buffer " + D.name);
    auto src = [&](int k) {
      const PlanBuf &S = bufs_[op.srcbuf[k]];
      if (!S.ptr) throw PlanError(CCLR_EINVAL, "perm on an unbound buffer " + S.name);
      return (const c128 *)S.ptr;
    };
    cudaError_t e = cudaSuccess;
    switch (op.special) {
      case 1: e = layout_unpack_rows(st_, src(0), D.ptr, op.sp_n, op.sp_len); break;
      case 2: e = layout_unpack_cols(st_, src(0), D.ptr, op.sp_len, op.sp_o); break;
      case 3: e = layout_unpack_ring(st_, src(0), D.ptr, op.sp_n, op.sp_o); break;
      case 4: e = layout_transpose_pair(st_, src(0), D.ptr, op.sp_len, op.sp_o); break;
      default:   // sources in statement order: x2, Y, Y, Q, Q, Z, Z, Z, Z
        e = layout_final_pack(st_, D.ptr, src(0), scalars_[0], src(1), src(3), src(5), op.sp_n, op.sp_o);
    }
    cuda_check(e, "layout(" + D.name + ")");
  } else {
    PermArgs args = op.args;
    const PlanBuf &D = bufs_[op.dst];
    if (!D.ptr) throw PlanError(CCLR_EINVAL, "perm on an unbound buffer " + D.name);
    args.dst = D.ptr + op.dstoff;
    for (int k = 0; k < args.nsrc; ++k) {
      const PlanBuf &S = bufs_[op.srcbuf[k]];
      if (!S.ptr) throw PlanError(CCLR_EINVAL, "perm on an unbound buffer " + S.name);
      args.src[k].ptr = S.ptr;
      if (op.src_scalar[k] >= 0) args.src[k].coef = scalars_[op.src_scalar[k]];
    }
    cuda_check(permute(st_, args), "permute(" + D.name + ")");
  }
}
