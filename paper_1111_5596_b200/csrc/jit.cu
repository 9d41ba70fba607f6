// jit.cu -- run-time expressions (second step): a lattice expression given as text is parsed,
// type-checked, written out as a node type of the expression layer (expr.cuh), compiled ONCE with NVRTC for sm_100a
// into a kernel of its own and kept in a cache keyed by the expression -- the scheme of the paper ("the tree parser
// generates the CUDA kernel code for the expression, which is then JIT-compiled ... each expression is compiled only
// once"), with the paper's PETE tree replaced by a small grammar and its code generator by the
// template layer the build-time expressions already use.  Host code only: the kernels come out of NVRTC.
//
//   expr   := term { ('+'|'-') term }
//   term   := factor { '*' factor }
//   factor := '-' factor | 'adj' '(' expr ')' | 'trace' '(' expr ')' | 'real' '(' expr ')' | 'imag' '(' expr ')'
//           | 'norm2' '(' expr ')' | 'inner' '(' expr ',' expr ')'
//           | 'shift' '(' expr ',' ('+'|'-') DIGIT ')' | '(' expr ')' | leaf
//   leaf   := 'f' DIGIT [ '[' DIGIT ']' ]     field argument DIGIT: matrix [slot] of a colour-matrix or gauge field (slot:
//                                             link of a gauge field, default 0), or the spinor of a fermion field
//           | 's' DIGIT                       real scalar argument DIGIT
//           | NUMBER                          decimal literal (2, 0.5, 1.5e-3): a real constant, part of the expression's type
// Value kinds: matrix (3x3 complex), complex, real, spinor (4 spin x 3 colour).  s -> real, adj keeps the kind (not
// defined on spinors), trace: matrix -> complex, real/imag: complex -> real, norm2: spinor -> real, inner: two spinors ->
// complex (the first conjugated), shift keeps the kind (shift(e, +mu)(x) = e(x + mu), A3), '+' and '-' need equal kinds,
// the unary minus keeps the kind and binds tighter than '*',
// '*': matrix*matrix, matrix*spinor (colour rotation of every spin component), real*anything, anything*real,
// complex*complex, complex*spinor.
//
// NVRTC is loaded with dlopen at the first compilation (the library does not link it), the headers the generated
// translation unit includes are embedded in this object at build time (build.py -> jit_headers.inc), and the cubin is
// loaded with cudaLibraryLoadData: nothing is read from the file system at run time.
#include <dlfcn.h>
#include <nvrtc.h>

#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "expr.cuh"
#include "jit_headers.inc"   // kJitHeaderNames[], kJitHeaderSources[], kJitHeaderCount

namespace qdp {

// ---- parser -----------------------------------------------------------------------------------------------------
namespace {

struct Parsed {
    std::string type;   // node type of expr.cuh
    int kind;           // JIT_MAT / JIT_CPLX / JIT_REAL
};

struct Parser {
    const char* s;
    const int* ncomp;   // components per site of the field arguments
    int nfields, nscalars;
    bool has_shift = false;
    unsigned fields_used = 0;
    std::string err;

    void skip() { while (*s == ' ' || *s == '\t' || *s == '\n') s++; }
    bool eat(char c) { skip(); if (*s == c) { s++; return true; } return false; }
    bool word(const char* w) {
        skip();
        size_t n = strlen(w);
        if (strncmp(s, w, n) == 0 && !((s[n] >= 'a' && s[n] <= 'z') || (s[n] >= '0' && s[n] <= '9'))) { s += n; return true; }
        return false;
    }
    bool fail(const std::string& m) { if (err.empty()) err = m + " at '" + std::string(s).substr(0, 16) + "'"; return false; }
    bool digit(int& d) { skip(); if (*s < '0' || *s > '9') return fail("digit expected"); d = *s++ - '0'; return true; }

    bool expr(Parsed& out) {
        if (!term(out)) return false;
        for (;;) {
            const bool plus = eat('+');
            if (!plus && !eat('-')) return true;
            Parsed r;
            if (!term(r)) return false;
            if (r.kind != out.kind) return fail("'+' and '-' need operands of the same kind (matrix, spinor, complex or real)");
            out.type = std::string(plus ? "Sum<" : "Diff<") + out.type + ", " + r.type + " >";
        }
    }
    bool term(Parsed& out) {
        if (!factor(out)) return false;
        while (eat('*')) {
            Parsed r;
            if (!factor(r)) return false;
            if (out.kind == JIT_MAT && (r.kind == JIT_MAT || r.kind == JIT_SPINOR)) { out.type = "Product<" + out.type + ", " + r.type + " >"; out.kind = r.kind; }
            else if (out.kind == JIT_REAL) { out.type = "Product<" + out.type + ", " + r.type + " >"; out.kind = r.kind; }
            else if (r.kind == JIT_REAL) {
                // real factors go first where expr.cuh has no mirror image of v_mul(real, x)
                out.type = out.kind == JIT_CPLX ? "Product<" + r.type + ", " + out.type + " >" : "Product<" + out.type + ", " + r.type + " >";
            }
            else if (out.kind == JIT_CPLX && (r.kind == JIT_CPLX || r.kind == JIT_SPINOR)) { out.type = "Product<" + out.type + ", " + r.type + " >"; out.kind = r.kind; }
            else if (out.kind == JIT_SPINOR && r.kind == JIT_CPLX) { out.type = "Product<" + r.type + ", " + out.type + " >"; }
            else return fail("'*' is not defined for these operand kinds");
        }
        return true;
    }
    bool unary(const char* node, Parsed& out, int want, int gives, const char* what) {
        if (!eat('(')) return fail("'(' expected");
        if (!expr(out)) return false;
        if (!eat(')')) return fail("')' expected");
        if (want >= 0 && out.kind != want) return fail(what);
        out.type = std::string(node) + "<" + out.type + " >";
        if (gives >= 0) out.kind = gives;
        return true;
    }
    bool factor(Parsed& out) {
        if (eat('-')) {
            if (!factor(out)) return false;
            out.type = "Neg<" + out.type + " >";
            return true;
        }
        if (word("adj")) {
            if (!unary("Adjoint", out, -1, -1, "")) return false;
            if (out.kind == JIT_SPINOR) return fail("adj() of a spinor is not defined");
            return true;
        }
        if (word("norm2")) return unary("Norm2", out, JIT_SPINOR, JIT_REAL, "norm2() takes a spinor");
        if (word("inner")) {
            Parsed b;
            if (!eat('(')) return fail("'(' expected");
            if (!expr(out)) return false;
            if (!eat(',')) return fail("',' expected");
            if (!expr(b)) return false;
            if (!eat(')')) return fail("')' expected");
            if (out.kind != JIT_SPINOR || b.kind != JIT_SPINOR) return fail("inner() takes two spinors");
            out.type = "Inner<" + out.type + ", " + b.type + " >";
            out.kind = JIT_CPLX;
            return true;
        }
        if (word("trace")) return unary("Trace", out, JIT_MAT, JIT_CPLX, "trace() takes a matrix");
        if (word("real")) return unary("Real", out, JIT_CPLX, JIT_REAL, "real() takes a complex number");
        if (word("imag")) return unary("Imag", out, JIT_CPLX, JIT_REAL, "imag() takes a complex number");
        if (word("shift")) {
            if (!eat('(')) return fail("'(' expected");
            if (!expr(out)) return false;
            if (!eat(',')) return fail("',' expected");
            skip();
            int sign = 0, mu = 0;
            if (*s == '+') sign = 1; else if (*s == '-') sign = -1; else return fail("'+' or '-' expected");
            s++;
            if (!digit(mu)) return false;
            if (mu > 3) return fail("direction must be 0..3");
            if (!eat(')')) return fail("')' expected");
            out.type = "Shifted<" + out.type + ", " + std::to_string(mu) + ", " + (sign > 0 ? "+1" : "-1") + ">";
            has_shift = true;
            return true;
        }
        if (eat('(')) {
            if (!expr(out)) return false;
            if (!eat(')')) return fail("')' expected");
            return true;
        }
        skip();
        if (*s == 'f') {
            s++;
            int k = 0, slot = 0;
            if (!digit(k)) return false;
            if (k >= nfields) return fail("field argument out of range");
            if (ncomp[k] == 12) {
                if (*s == '[') return fail("a fermion field has no slots");
                out.type = "F<" + std::to_string(k) + ">";
                out.kind = JIT_SPINOR;
                fields_used |= 1u << k;
                return true;
            }
            if (*s == '[') { s++; if (!digit(slot)) return false; if (!eat(']')) return fail("']' expected"); }
            if (ncomp[k] != 9 && ncomp[k] != 36) return fail("field arguments must be colour matrices, gauge fields or fermions");
            if (slot >= ncomp[k] / 9) return fail("slot out of range");
            out.type = "M<" + std::to_string(k) + ", " + std::to_string(ncomp[k]) + ", " + std::to_string(slot) + ">";
            out.kind = JIT_MAT;
            fields_used |= 1u << k;
            return true;
        }
        if (*s == 's') {
            s++;
            int k = 0;
            if (!digit(k)) return false;
            if (k >= nscalars) return fail("scalar argument out of range");
            out.type = "Sc<" + std::to_string(k) + ">";
            out.kind = JIT_REAL;
            return true;
        }
        if ((*s >= '0' && *s <= '9') || (*s == '.' && s[1] >= '0' && s[1] <= '9')) {
            // digits [. digits] [e [+-] digits]; scanned here so that the accepted spellings do not depend on strtod's
            // extras (hex floats, "inf", locale)
            const char* b = s;
            while (*s >= '0' && *s <= '9') s++;
            if (*s == '.') { s++; while (*s >= '0' && *s <= '9') s++; }
            if (*s == 'e' || *s == 'E') {
                const char* m = s + 1;
                if (*m == '+' || *m == '-') m++;
                if (*m < '0' || *m > '9') return fail("digits expected in the exponent");
                while (*m >= '0' && *m <= '9') m++;
                s = m;
            }
            if ((*s >= 'a' && *s <= 'z') || (*s >= 'A' && *s <= 'Z') || *s == '.') return fail("malformed number");
            const double v = strtod(std::string(b, s).c_str(), nullptr);
            unsigned long long bits;
            memcpy(&bits, &v, sizeof bits);
            char buf[40];
            snprintf(buf, sizeof buf, "Lit<0x%016llxull>", bits);
            out.type = buf;
            out.kind = JIT_REAL;
            return true;
        }
        return fail("operand expected");
    }
};

}  // namespace

int jit_parse(const char* text, const int* ncomp, int nfields, int nscalars, JitExpr* out, std::string* err) {
    if (!text || nfields < 0 || nfields > 4 || nscalars < 0 || nscalars > 4) { if (err) *err = "bad argument"; return -1; }
    Parser p;
    p.s = text; p.ncomp = ncomp; p.nfields = nfields; p.nscalars = nscalars;
    Parsed r;
    bool ok = p.expr(r);
    if (ok) { p.skip(); if (*p.s) ok = p.fail("unexpected input"); }
    if (!ok) { if (err) *err = p.err; return -1; }
    out->type = r.type; out->kind = r.kind; out->has_shift = p.has_shift; out->fields_used = p.fields_used;
    return 0;
}

// ---- NVRTC, loaded on demand ---------------------------------------------------------------------------------------
namespace {

struct Nvrtc {
    void* h = nullptr;
    decltype(&nvrtcCreateProgram) create = nullptr;
    decltype(&nvrtcCompileProgram) compile = nullptr;
    decltype(&nvrtcGetCUBINSize) cubin_size = nullptr;
    decltype(&nvrtcGetCUBIN) cubin = nullptr;
    decltype(&nvrtcGetProgramLogSize) log_size = nullptr;
    decltype(&nvrtcGetProgramLog) log = nullptr;
    decltype(&nvrtcDestroyProgram) destroy = nullptr;
    bool load(std::string* err) {
        if (h) return true;
        const char* names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"};
        for (const char* n : names) if ((h = dlopen(n, RTLD_NOW | RTLD_LOCAL))) break;
        if (!h) { *err = "cannot load libnvrtc (needed for run-time expressions)"; return false; }
#define QDP_SYM(field, name) field = reinterpret_cast<decltype(field)>(dlsym(h, #name)); if (!field) { *err = "libnvrtc lacks " #name; h = nullptr; return false; }
        QDP_SYM(create, nvrtcCreateProgram) QDP_SYM(compile, nvrtcCompileProgram) QDP_SYM(cubin_size, nvrtcGetCUBINSize)
        QDP_SYM(cubin, nvrtcGetCUBIN) QDP_SYM(log_size, nvrtcGetProgramLogSize) QDP_SYM(log, nvrtcGetProgramLog)
        QDP_SYM(destroy, nvrtcDestroyProgram)
#undef QDP_SYM
        return true;
    }
};

struct Compiled {
    std::vector<char> cubin;
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kernel = nullptr;
};

std::mutex g_jit_mutex;
Nvrtc g_nvrtc;
std::map<std::string, Compiled> g_jit_cache;
long long g_jit_compilations = 0;

}  // namespace

std::string jit_source(const JitExpr& e, int prec, bool sum) {
    std::string src = "#include \"expr.cuh\"\nusing namespace qdp;\nusing namespace qdp::ex;\n";
    src += std::string("typedef ") + (prec ? "double" : "float") + " T_;\n";
    src += "typedef " + e.type + " E_;\n";
    if (sum)
        src += std::string("extern \"C\" __global__ void __launch_bounds__(128, ") + (prec ? "2" : "4") +
               ") qdp_jit_kernel(Geom g, Args a, int subset, ReduceBuf rb) { sumv_body<T_, E_>(g, a, subset, rb); }\n";
    else
        src += "extern \"C\" __global__ void __launch_bounds__(128) qdp_jit_kernel(Geom g, Args a, Vec2<T_>::type* dst, int nd, int cd, int subset) "
               "{ assign_body<T_, E_>(g, a, dst, nd, cd, subset); }\n";
    return src;
}

// compiles (or finds) the kernel of (expression type, precision, assign | sum); *cubin_out (optional) receives the image
static int jit_get(const JitExpr& e, int prec, bool sum, bool load, Compiled** out, std::string* err) {
    const std::string key = std::string(prec ? "d" : "f") + (sum ? "S:" : "A:") + e.type;
    std::lock_guard<std::mutex> lock(g_jit_mutex);
    auto it = g_jit_cache.find(key);
    if (it == g_jit_cache.end()) {
        if (!g_nvrtc.load(err)) return -1;
        const std::string src = jit_source(e, prec, sum);
        nvrtcProgram prog;
        if (g_nvrtc.create(&prog, src.c_str(), "qdp_expr_jit.cu", kJitHeaderCount, kJitHeaderSources, kJitHeaderNames) != NVRTC_SUCCESS) {
            *err = "nvrtcCreateProgram failed";
            return -1;
        }
#ifdef QDP_BOUNDS_CHECK   // the bounds-checked build validates the site addresses of its run-time kernels too
        const char* opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "-DQDP_BOUNDS_CHECK"};
#else
        const char* opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo"};
#endif
        const nvrtcResult rc = g_nvrtc.compile(prog, (int)(sizeof(opts) / sizeof(opts[0])), opts);
        if (rc != NVRTC_SUCCESS) {
            size_t n = 0;
            g_nvrtc.log_size(prog, &n);
            std::string log(n, '\0');
            if (n) g_nvrtc.log(prog, &log[0]);
            *err = "NVRTC: " + log.substr(0, 600);
            g_nvrtc.destroy(&prog);
            return -1;
        }
        Compiled c;
        size_t n = 0;
        g_nvrtc.cubin_size(prog, &n);
        c.cubin.resize(n);
        g_nvrtc.cubin(prog, c.cubin.data());
        g_nvrtc.destroy(&prog);
        g_jit_compilations++;
        it = g_jit_cache.emplace(key, std::move(c)).first;
    }
    Compiled& c = it->second;
    if (load && !c.kernel) {
        cudaError_t ce = cudaLibraryLoadData(&c.lib, c.cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
        if (ce == cudaSuccess) ce = cudaLibraryGetKernel(&c.kernel, c.lib, "qdp_jit_kernel");
        if (ce != cudaSuccess) { *err = std::string("loading the compiled expression failed: ") + cudaGetErrorString(ce); c.kernel = nullptr; return -1; }
    }
    *out = &c;
    return 0;
}

long long jit_compilations() {
    std::lock_guard<std::mutex> lock(g_jit_mutex);
    return g_jit_compilations;
}

// compile only (no device needed): used by the CPU tests and to warm the cache; *cubin_bytes receives the image size
int jit_compile_only(const JitExpr& e, int prec, bool sum, size_t* cubin_bytes, std::string* err) {
    Compiled* c = nullptr;
    if (jit_get(e, prec, sum, false, &c, err) != 0) return -1;
    if (cubin_bytes) *cubin_bytes = c->cubin.size();
    return 0;
}

cudaError_t jit_launch_assign(const JitExpr& e, int prec, const Geom& g, const ex::Args& a, void* dst, int nd, int cd, int subset,
                              cudaStream_t st, std::string* err) {
    Compiled* c = nullptr;
    if (jit_get(e, prec, false, true, &c, err) != 0) return cudaErrorUnknown;
    const int items = subset == 0 ? 2 * ((g.Vh + 31) & ~31) : g.Vh;
    Geom gg = g;
    ex::Args aa = a;
    void* args[] = {&gg, &aa, &dst, &nd, &cd, &subset};
    cudaError_t ce = cudaLaunchKernel((const void*)c->kernel, dim3((items + 127) / 128), dim3(128), args, 0, st);
    g_launch_count++;
    return ce;
}

cudaError_t jit_launch_sum(const JitExpr& e, int prec, const Geom& g, const ex::Args& a, int subset, const ReduceBuf& rb,
                           cudaStream_t st, std::string* err) {
    Compiled* c = nullptr;
    if (jit_get(e, prec, true, true, &c, err) != 0) return cudaErrorUnknown;
    const int items = subset == 0 ? 2 * g.Vhp : g.Vh;
    int grid = (items + 127) / 128;
    const int cap = device_sm_count() * (prec ? 2 : 4);
    if (grid > cap) grid = cap;
    Geom gg = g;
    ex::Args aa = a;
    ReduceBuf r = rb;
    void* args[] = {&gg, &aa, &subset, &r};
    cudaError_t ce = cudaLaunchKernel((const void*)c->kernel, dim3(grid), dim3(128), args, 0, st);
    g_launch_count++;
    return ce;
}

}  // namespace qdp
