// expr.cu -- NEXT-2: the user-extensible fused element-wise front end.
//
// The paper's second contribution is that whole-array arithmetic written by the user
//     soax.posArr(0) = soax.velArr(1) - soax.velArr(2);
// is fused by expression templates into ONE loop / ONE kernel without temporaries (PAPER.md:322, 360-366,
// "loop fusion"), and that a user functor can be applied to the arrays.  C++ expression
// templates cannot cross a C ABI, so the same idea is restated for B200: the user hands over the PROGRAM TEXT
//     "vel = fma(float(dt), float(-(pos - 0.5)), vel); pos = wrap(fma(dt, double(vel), pos))"
// soax_expr_compile type-checks it against the layout, generates one CUDA kernel for it -- shaped exactly like the
// hand-written step kernels: each thread owns 4 consecutive particles, every field array that the program reads is
// loaded once with a 128/256-bit access, every array it assigns is stored once -- and compiles that kernel with
// NVRTC for sm_100a (-fmad=false: the arithmetic contract of DESIGN.md holds for generated code too).
// soax_expr_run launches it.  Statements run in order per particle and later statements see earlier assignments,
// so a whole integrator step is one fused pass.  Nothing is interpreted at run time and nothing runs on the host.
//
// Language (include/soax.h has the user-level description):
//   program := stmt { ';' stmt } [';']          stmt := target ('=' | '+=' | '-=' | '*=' | '/=') expr
//   target  := field | field '[' c ']'          a dim-3 field without index means "for c = 0, 1, 2"
//   expr    := C arithmetic with + - * / unary -, comparisons, '&' on integers, parentheses, numbers, named scalars,
//              field reads, and calls: fma sqrt abs min max floor wrap float double select
#include <dlfcn.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <mutex>
#include <string>
#include <vector>

#include "common.cuh"
#include "expr.hpp"
#include "ops.hpp"

namespace soax {
namespace {

thread_local std::string g_expr_error;

// ---- types ------------------------------------------------------------------------------------------------------
enum Ty { T_I32 = SOAX_I32, T_I64 = SOAX_I64, T_U8 = SOAX_U8, T_F32 = SOAX_F32, T_F64 = SOAX_F64, T_BOOL = 16, T_ILIT = 17 };
bool is_float(int t) { return t == T_F32 || t == T_F64; }
bool is_int(int t) { return t == T_I32 || t == T_I64 || t == T_U8 || t == T_ILIT; }
const char* c_name(int t) {
    switch (t) {
        case T_I32: return "int";
        case T_I64: return "long long";
        case T_U8: return "unsigned char";
        case T_F32: return "float";
        case T_F64: return "double";
        case T_BOOL: return "bool";
        default: return "long long";
    }
}

struct ParseError {
    std::string msg;
    size_t pos;
};

// ---- tokens -----------------------------------------------------------------------------------------------------
struct Tok {
    enum Kind { END, NUM, INT, ID, OP } kind = END;
    std::string text;
    double num = 0.0;
    long long ival = 0;
    size_t pos = 0;
};

std::vector<Tok> tokenize(const std::string& s) {
    std::vector<Tok> out;
    size_t i = 0;
    while (i < s.size()) {
        const char ch = s[i];
        if (ch == ' ' || ch == '\t' || ch == '\n' || ch == '\r') { ++i; continue; }
        Tok t;
        t.pos = i;
        if ((ch >= '0' && ch <= '9') || (ch == '.' && i + 1 < s.size() && s[i + 1] >= '0' && s[i + 1] <= '9')) {
            char* end = nullptr;
            t.num = std::strtod(s.c_str() + i, &end);
            const size_t len = (size_t)(end - (s.c_str() + i));
            t.text = s.substr(i, len);
            const bool integral = t.text.find_first_of(".eExXpP") == std::string::npos;
            t.kind = integral ? Tok::INT : Tok::NUM;
            if (integral) t.ival = std::strtoll(t.text.c_str(), nullptr, 10);
            i += len;
        } else if ((ch >= 'a' && ch <= 'z') || (ch >= 'A' && ch <= 'Z') || ch == '_') {
            size_t j = i;
            while (j < s.size() && ((s[j] >= 'a' && s[j] <= 'z') || (s[j] >= 'A' && s[j] <= 'Z') || (s[j] >= '0' && s[j] <= '9') || s[j] == '_')) ++j;
            t.kind = Tok::ID;
            t.text = s.substr(i, j - i);
            i = j;
        } else {
            static const char* two[] = {"+=", "-=", "*=", "/=", "<=", ">=", "==", "!="};
            t.kind = Tok::OP;
            bool found = false;
            for (const char* op : two)
                if (s.compare(i, 2, op) == 0) { t.text = op; i += 2; found = true; break; }
            if (!found) {
                if (!std::strchr("+-*/()[],;=<>&|", ch)) throw ParseError{std::string("unexpected character '") + ch + "'", i};
                t.text = std::string(1, ch);
                ++i;
            }
        }
        out.push_back(t);
    }
    Tok e;
    e.pos = s.size();
    out.push_back(e);
    return out;
}

// ---- typed expression tree, rendered to CUDA C++ as it is built ------------------------------------------------------
struct Val {
    std::string code;  // a parenthesised C++ expression over the per-particle locals x<C> and the scalars a.s[k]
    int ty;
    long long ilit = 0;
};

struct Program {
    const ExprLayoutInfo* L;
    std::vector<std::string> scalar_names;
    std::vector<bool> read_first;  // component is read before (or without) being assigned: must be loaded
    std::vector<bool> assigned;    // component is assigned: must be stored
    std::vector<bool> touched;
    std::string body;              // statements over the locals, one particle
    bool is_sum = false;           // the program is ONE expression whose per-particle value is summed in double
    bool is_mask = false;          // the program is ONE condition whose per-particle truth value is written as a byte
};

std::string hex_double(double v) {
    char buf[64];
    if (std::isinf(v) || std::isnan(v)) throw ParseError{"non-finite literal", 0};
    std::snprintf(buf, sizeof buf, "%a", v);
    return buf;
}

class Parser {
  public:
    Parser(const std::string& src, Program& prog) : toks_(tokenize(src)), P_(prog) {}

    void program() {
        while (peek().kind != Tok::END) {
            if (is_op(";")) { next(); continue; }
            statement();
            if (peek().kind != Tok::END && !is_op(";")) fail("expected ';' between statements");
        }
    }

    // a reduction program: one floating-point expression, summed over the particles in double
    void sum_expression() {
        Val v = expr();
        if (is_op(";")) next();
        if (peek().kind != Tok::END) fail("a sum program is a single expression");
        if (v.ty == T_ILIT) v = to_float(v, T_F64, 0);
        if (!is_float(v.ty)) fail("the summed expression must be a floating-point value (use float()/double())");
        P_.body += "        acc += (double)" + v.code + ";\n";
    }

    // a mask program: one condition (a comparison, or comparisons joined by '&' and '|'), stored as one byte per particle
    void mask_expression() {
        Val v = expr();
        if (is_op(";")) next();
        if (peek().kind != Tok::END) fail("a mask program is a single condition");
        if (v.ty != T_BOOL) fail("the mask expression must be a condition (a comparison, or comparisons joined by '&' / '|')");
        P_.body += "        mk[j] = " + v.code + " ? (unsigned char)1 : (unsigned char)0;\n";
    }

  private:
    std::vector<Tok> toks_;
    size_t at_ = 0;
    Program& P_;
    int vec_c_ = -1;  // component index substituted for un-indexed dim-3 fields in the statement being expanded
    int vec_dim_ = 0; // dimension of the target of that statement

    const Tok& peek() const { return toks_[at_]; }
    Tok next() { return toks_[at_++]; }
    bool is_op(const char* op) const { return peek().kind == Tok::OP && peek().text == op; }
    [[noreturn]] void fail(const std::string& m) const { throw ParseError{m, peek().pos}; }
    void expect(const char* op) {
        if (!is_op(op)) fail(std::string("expected '") + op + "'");
        next();
    }

    int find_field(const std::string& name) const {
        for (int f = 0; f < P_.L->nfields; ++f)
            if (name == P_.L->fname[f]) return f;
        return -1;
    }
    int find_scalar(const std::string& name) const {
        for (size_t k = 0; k < P_.scalar_names.size(); ++k)
            if (name == P_.scalar_names[k]) return (int)k;
        return -1;
    }

    // field reference -> global component index; handles [c] and the vector form
    int component(const Tok& id, int f) {
        const int dim = P_.L->fdim[f];
        int c = 0;
        if (is_op("[")) {
            next();
            if (peek().kind != Tok::INT) fail("component index must be an integer literal");
            c = (int)next().ival;
            expect("]");
            if (c < 0 || c >= dim) throw ParseError{"component " + std::to_string(c) + " is outside field '" + id.text + "' of dimension " + std::to_string(dim) + " (PAPER.md:320)", id.pos};
        } else if (dim > 1) {
            if (vec_c_ < 0) throw ParseError{"field '" + id.text + "' has " + std::to_string(dim) + " components: index it, or assign to a vector field", id.pos};
            if (dim != vec_dim_) throw ParseError{"vector statement mixes fields of different dimension at '" + id.text + "'", id.pos};
            c = vec_c_;
        }
        return P_.L->fbegin[f] + c;
    }

    static std::string local(int comp) { return "x" + std::to_string(comp); }

    // ---- statements ------------------------------------------------------------------------------------------------
    void statement() {
        const size_t start = at_;
        const Tok id = peek();
        if (id.kind != Tok::ID) fail("expected a field name at the start of a statement");
        const int f = find_field(id.text);
        if (f < 0) fail("unknown field '" + id.text + "'");
        // vector form: target is an un-indexed field of dimension > 1
        const bool vector_form = P_.L->fdim[f] > 1 && !(toks_[at_ + 1].kind == Tok::OP && toks_[at_ + 1].text == "[");
        const int reps = vector_form ? P_.L->fdim[f] : 1;
        size_t end = at_;
        vec_dim_ = P_.L->fdim[f];
        for (int r = 0; r < reps; ++r) {
            at_ = start;
            vec_c_ = vector_form ? r : -1;
            one_statement();
            end = at_;
        }
        vec_c_ = -1;
        at_ = end;
    }

    void one_statement() {
        const Tok id = next();
        const int f = find_field(id.text);
        const int comp = component(id, f);
        const int ty = P_.L->cdtype[comp];
        if (!is_float(ty)) throw ParseError{"assignment to integer field '" + id.text + "' is not supported", id.pos};
        if (peek().kind != Tok::OP) fail("expected an assignment operator");
        const std::string op = next().text;
        if (op != "=" && op != "+=" && op != "-=" && op != "*=" && op != "/=") throw ParseError{"expected '=', '+=', '-=', '*=' or '/='", toks_[at_ - 1].pos};
        if (op != "=") mark_read(comp);
        Val rhs = expr();
        if (rhs.ty == T_ILIT) rhs = to_float(rhs, ty, id.pos);  // an integer literal takes the type of the target
        if (!is_float(rhs.ty)) fail("the right-hand side must be a floating-point value (use float()/double())");
        std::string value = rhs.code;
        if (op != "=") {  // a op= b  is  a = (T)(a op b)  with the usual promotion of a and b
            Val lhs{local(comp), ty};
            value = binary(op.substr(0, 1), lhs, rhs, id.pos).code;
        }
        P_.body += "        " + local(comp) + " = (" + c_name(ty) + ")" + value + ";\n";
        P_.assigned[comp] = true;
        P_.touched[comp] = true;
    }

    void mark_read(int comp) {
        if (!P_.assigned[comp]) P_.read_first[comp] = true;
        P_.touched[comp] = true;
    }

    // ---- expressions: comparison < additive < multiplicative < unary < primary ------------------------------------------
    // precedence (lowest first, Python's): comparison, '|', '&', additive, multiplicative, unary.  '&' and '|' bind TIGHTER
    // than comparisons, so conditions are joined as (a < b) & (c >= d) -- with the parentheses.
    Val expr() {
        Val a = bitor_();
        while (is_op("<") || is_op("<=") || is_op(">") || is_op(">=") || is_op("==") || is_op("!=")) {
            const Tok op = next();
            Val b = bitor_();
            a = compare(op.text, a, b, op.pos);
        }
        return a;
    }
    Val bitor_() {
        Val a = bitand_();
        while (is_op("|")) {
            const Tok op = next();
            Val b = bitand_();
            if (a.ty != T_BOOL || b.ty != T_BOOL) throw ParseError{"'|' joins two conditions (parenthesised comparisons)", op.pos};
            a = Val{"(" + a.code + " || " + b.code + ")", T_BOOL};
        }
        return a;
    }
    Val bitand_() {
        Val a = additive();
        while (is_op("&")) {
            const Tok op = next();
            Val b = additive();
            if (a.ty == T_BOOL && b.ty == T_BOOL) { a = Val{"(" + a.code + " && " + b.code + ")", T_BOOL}; continue; }
            if (!is_int(a.ty) || !is_int(b.ty)) throw ParseError{"'&' needs integer operands or two conditions", op.pos};
            const int ty = a.ty == T_ILIT ? b.ty : a.ty;
            if (a.ty != T_ILIT && b.ty != T_ILIT && a.ty != b.ty) throw ParseError{"'&' between different integer types", op.pos};
            a = Val{"((" + std::string(c_name(ty)) + ")(" + a.code + " & " + b.code + "))", ty == T_ILIT ? T_I64 : ty};
        }
        return a;
    }
    Val additive() {
        Val a = multiplicative();
        while (is_op("+") || is_op("-")) {
            const Tok op = next();
            Val b = multiplicative();
            a = binary(op.text, a, b, op.pos);
        }
        return a;
    }
    Val multiplicative() {
        Val a = unary();
        while (is_op("*") || is_op("/")) {
            const Tok op = next();
            Val b = unary();
            a = binary(op.text, a, b, op.pos);
        }
        return a;
    }
    Val unary() {
        if (is_op("-")) {
            const Tok op = next();
            Val a = unary();
            if (a.ty == T_ILIT) return Val{"(-" + a.code + ")", T_ILIT, -a.ilit};
            if (!is_float(a.ty)) throw ParseError{"unary '-' needs a floating-point operand", op.pos};
            return Val{"(-" + a.code + ")", a.ty};
        }
        if (is_op("+")) { next(); return unary(); }
        return primary();
    }

    // usual arithmetic conversions restricted to float/double: integer LITERALS adapt to the other operand's type
    Val to_float(const Val& v, int ty, size_t pos) const {
        if (v.ty == ty) return v;
        if (v.ty == T_ILIT) return Val{"(" + std::string(ty == T_F32 ? "(float)" : "") + hex_double((double)v.ilit) + ")", ty};
        if (is_float(v.ty)) return Val{"((" + std::string(c_name(ty)) + ")" + v.code + ")", ty};
        throw ParseError{"integer field in floating-point arithmetic: convert it with float() or double()", pos};
    }
    static int promote(const Val& a, const Val& b) {
        if (a.ty == T_F64 || b.ty == T_F64) return T_F64;
        if (a.ty == T_F32 || b.ty == T_F32) return T_F32;
        return T_F64;  // two integer literals
    }
    Val binary(const std::string& op, const Val& a, const Val& b, size_t pos) const {
        if ((!is_float(a.ty) && a.ty != T_ILIT) || (!is_float(b.ty) && b.ty != T_ILIT))
            throw ParseError{"'" + op + "' needs floating-point operands (convert integer fields with float()/double())", pos};
        const int ty = promote(a, b);
        const Val x = to_float(a, ty, pos), y = to_float(b, ty, pos);
        return Val{"(" + x.code + " " + op + " " + y.code + ")", ty};
    }
    Val compare(const std::string& op, const Val& a, const Val& b, size_t pos) const {
        if (is_int(a.ty) && is_int(b.ty)) {
            if (a.ty != T_ILIT && b.ty != T_ILIT && a.ty != b.ty) throw ParseError{"comparison between different integer types", pos};
            return Val{"(" + a.code + " " + op + " " + b.code + ")", T_BOOL};
        }
        if (a.ty == T_BOOL || b.ty == T_BOOL) throw ParseError{"a comparison result cannot be compared again", pos};
        const int ty = promote(a, b);
        const Val x = to_float(a, ty, pos), y = to_float(b, ty, pos);
        return Val{"(" + x.code + " " + op + " " + y.code + ")", T_BOOL};
    }

    std::vector<Val> call_args(size_t nargs, const Tok& fn) {
        expect("(");
        std::vector<Val> a;
        if (!is_op(")")) {
            a.push_back(expr());
            while (is_op(",")) { next(); a.push_back(expr()); }
        }
        expect(")");
        if (a.size() != nargs) throw ParseError{fn.text + "() takes " + std::to_string(nargs) + " argument(s)", fn.pos};
        return a;
    }

    Val primary() {
        const Tok t = next();
        if (t.kind == Tok::NUM) return Val{"(" + hex_double(t.num) + ")", T_F64};
        if (t.kind == Tok::INT) return Val{"(" + std::to_string(t.ival) + "ll)", T_ILIT, t.ival};
        if (t.kind == Tok::OP && t.text == "(") {
            Val v = expr();
            expect(")");
            return v;
        }
        if (t.kind != Tok::ID) throw ParseError{"expected a value", t.pos};
        if (is_op("(")) return call(t);
        const int f = find_field(t.text);
        if (f >= 0) {
            const int comp = component(t, f);
            mark_read(comp);
            return Val{local(comp), P_.L->cdtype[comp]};
        }
        const int k = find_scalar(t.text);
        if (k >= 0) return Val{"a.s[" + std::to_string(k) + "]", T_F64};
        throw ParseError{"unknown name '" + t.text + "' (neither a field of the layout nor a declared scalar)", t.pos};
    }

    Val call(const Tok& fn) {
        const std::string& n = fn.text;
        if (n == "float" || n == "double") {
            const int ty = n == "float" ? T_F32 : T_F64;
            Val v = call_args(1, fn)[0];
            if (v.ty == T_BOOL) throw ParseError{"cannot convert a comparison result; use select()", fn.pos};
            if (v.ty == T_ILIT) return to_float(v, ty, fn.pos);
            return Val{"((" + std::string(c_name(ty)) + ")" + v.code + ")", ty};
        }
        if (n == "cell") {  // a10: the particle's cell index on a G^3 grid, bit-equal to soax_bin_permute's
            expect("(");
            if (peek().kind != Tok::INT) fail("cell(G): G must be an integer literal");
            const long long G = next().ival;
            expect(")");
            if (G < 1 || G > 64 || (G & (G - 1)) != 0) throw ParseError{"cell(G): G must be a power of two, 1 <= G <= 64", fn.pos};
            const int f = find_field("pos");
            if (f < 0 || P_.L->fdim[f] != 3 || P_.L->cdtype[P_.L->fbegin[f]] != T_F64) throw ParseError{"cell(G) needs a field pos of three doubles", fn.pos};
            const int c0 = P_.L->fbegin[f];
            for (int c = 0; c < 3; ++c) mark_read(c0 + c);
            return Val{"soax_cell(" + local(c0) + ", " + local(c0 + 1) + ", " + local(c0 + 2) + ", " + std::to_string(G) + ")", T_I32};
        }
        if (n == "select") {
            std::vector<Val> a = call_args(3, fn);
            if (a[0].ty != T_BOOL) throw ParseError{"select(cond, a, b): cond must be a comparison", fn.pos};
            const int ty = promote(a[1], a[2]);
            const Val x = to_float(a[1], ty, fn.pos), y = to_float(a[2], ty, fn.pos);
            return Val{"(" + a[0].code + " ? " + x.code + " : " + y.code + ")", ty};
        }
        struct Fn { const char* name; int nargs; const char* f32; const char* f64; };
        static const Fn fns[] = {{"fma", 3, "fmaf", "fma"},   {"sqrt", 1, "sqrtf", "sqrt"}, {"abs", 1, "fabsf", "fabs"},
                                 {"min", 2, "fminf", "fmin"}, {"max", 2, "fmaxf", "fmax"}, {"floor", 1, "floorf", "floor"},
                                 {"wrap", 1, "soax_wrap01f", "soax_wrap01"}};
        for (const Fn& f : fns) {
            if (n != f.name) continue;
            std::vector<Val> a = call_args((size_t)f.nargs, fn);
            int ty = T_F32;
            bool any_float = false;
            for (const Val& v : a) {
                if (v.ty == T_F64) ty = T_F64;
                if (is_float(v.ty)) any_float = true;
                else if (v.ty != T_ILIT) throw ParseError{n + "() needs floating-point arguments", fn.pos};
            }
            if (!any_float) ty = T_F64;
            std::string code = std::string(ty == T_F32 ? f.f32 : f.f64) + "(";
            for (size_t i = 0; i < a.size(); ++i) code += (i ? ", " : "") + to_float(a[i], ty, fn.pos).code;
            return Val{"(" + code + "))", ty};
        }
        throw ParseError{"unknown function '" + n + "'", fn.pos};
    }
};

// ---- code generation --------------------------------------------------------------------------------------------------------
// Device prelude of every generated kernel: the vector access and wrap of the hand-written kernels, restated so that the
// generated translation unit is self-contained (NVRTC sees no project headers).
const char* kPrelude = R"PRE(
template <class T, int P> struct __align__(sizeof(T) * P > 32 ? 32 : sizeof(T) * P) Vec { T v[P]; };
template <class T, int P> __device__ __forceinline__ Vec<T, P> ld_vec(const T* p) {
    constexpr int B = sizeof(T) * P;
    Vec<T, P> r;
    unsigned* w = reinterpret_cast<unsigned*>(&r);
    if constexpr (B == 32) {
#ifndef SOAX_NO_256BIT
        asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]) : "l"(p));
#else
        asm volatile("ld.global.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(p));
        asm volatile("ld.global.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4+16];" : "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]) : "l"(p));
#endif
    } else if constexpr (B == 16) {
        asm volatile("ld.global.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(p));
    } else if constexpr (B == 8) {
        asm volatile("ld.global.L1::no_allocate.v2.b32 {%0,%1}, [%2];" : "=r"(w[0]), "=r"(w[1]) : "l"(p));
    } else {
        r = *reinterpret_cast<const Vec<T, P>*>(p);
    }
    return r;
}
template <class T, int P> __device__ __forceinline__ void st_vec(T* p, const Vec<T, P>& r) {
    constexpr int B = sizeof(T) * P;
    const unsigned* w = reinterpret_cast<const unsigned*>(&r);
    if constexpr (B == 32) {
#ifndef SOAX_NO_256BIT
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     :: "l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]) : "memory");
#else
        asm volatile("st.global.L1::no_allocate.v4.b32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
        asm volatile("st.global.L1::no_allocate.v4.b32 [%0+16], {%1,%2,%3,%4};" :: "l"(p), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]) : "memory");
#endif
    } else if constexpr (B == 16) {
        asm volatile("st.global.L1::no_allocate.v4.b32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
    } else if constexpr (B == 8) {
        asm volatile("st.global.L1::no_allocate.v2.b32 [%0], {%1,%2};" :: "l"(p), "r"(w[0]), "r"(w[1]) : "memory");
    } else {
        *reinterpret_cast<Vec<T, P>*>(p) = r;
    }
}
// wrap into [0,1): x - floor(x), a result of exactly 1 mapped to 0 (DESIGN.md Q3); floor-free fast path for -1 <= x < 2
__device__ __forceinline__ double soax_wrap01(double x) {
    double w;
    if (x >= -1.0 && x < 2.0) w = x + (x < 0.0 ? 1.0 : (x >= 1.0 ? -1.0 : 0.0));
    else w = x - floor(x);
    return w >= 1.0 ? 0.0 : w;
}
// a10: cell index on a G^3 grid, x slowest (Q11); pos*G is exact for G a power of two (Q16); truncation toward zero; an index
// outside the grid (a position outside [0,1): a precondition violation) is clamped into it, as soax_bin_permute does
__device__ __forceinline__ int soax_cell(double x0, double x1, double x2, int G) {
    const int i0 = min(max((int)(x0 * (double)G), 0), G - 1);
    const int i1 = min(max((int)(x1 * (double)G), 0), G - 1);
    const int i2 = min(max((int)(x2 * (double)G), 0), G - 1);
    return (i0 * G + i1) * G + i2;
}
__device__ __forceinline__ float soax_wrap01f(float x) {
    float w;
    if (x >= -1.0f && x < 2.0f) w = x + (x < 0.0f ? 1.0f : (x >= 1.0f ? -1.0f : 0.0f));
    else w = x - floorf(x);
    return w >= 1.0f ? 0.0f : w;
}
)PRE";

std::string generate(const Program& P) {
    const ExprLayoutInfo& L = *P.L;
    std::string s = "// generated by soax_expr_compile -- one fused pass, 4 particles per thread\n";
    s += kPrelude;
    s += "struct Args { void* p[" + std::to_string(L.ncomp) + "]; double s[" + std::to_string(P.scalar_names.empty() ? 1 : P.scalar_names.size()) + "]; };\n";
    s += std::string("template <int P> __device__ __forceinline__ ") + (P.is_sum ? "double" : "void") + " group(const Args& a, long long i0" +
         (P.is_mask ? ", unsigned char* mask" : "") + ") {\n";
    for (int c = 0; c < L.ncomp; ++c) {
        if (!P.touched[c]) continue;
        const std::string T = c_name(L.cdtype[c]), v = "v" + std::to_string(c);
        if (P.read_first[c]) s += "    Vec<" + T + ", P> " + v + " = ld_vec<" + T + ", P>(static_cast<const " + T + "*>(a.p[" + std::to_string(c) + "]) + i0);\n";
        else s += "    Vec<" + T + ", P> " + v + ";\n";
    }
    if (P.is_sum) s += "    double acc = 0.0;\n";
    if (P.is_mask) s += "    unsigned char mk[P];\n";
    s += "#pragma unroll\n    for (int j = 0; j < P; ++j) {\n";
    for (int c = 0; c < L.ncomp; ++c)
        if (P.touched[c]) s += "        " + std::string(c_name(L.cdtype[c])) + "& x" + std::to_string(c) + " = v" + std::to_string(c) + ".v[j];\n";
    s += P.body;
    s += "    }\n";
    for (int c = 0; c < L.ncomp; ++c)
        if (P.assigned[c]) {
            const std::string T = c_name(L.cdtype[c]);
            s += "    st_vec<" + T + ", P>(static_cast<" + T + "*>(a.p[" + std::to_string(c) + "]) + i0, v" + std::to_string(c) + ");\n";
        }
    if (P.is_sum) s += "    return acc;\n";
    if (P.is_mask)  // four mask bytes leave as one 32-bit store (mask + i0 is 4-byte aligned: i0 is a multiple of 4)
        s += "    if constexpr (P == 4) *reinterpret_cast<unsigned*>(mask + i0) = mk[0] | (mk[1] << 8) | (mk[2] << 16) | ((unsigned)mk[3] << 24);\n"
             "    else mask[i0] = mk[0];\n";
    s += "}\n";
    if (P.is_mask) {
        s += R"K(extern "C" __global__ void __launch_bounds__(512) soax_expr_kernel(const Args a, const long long n, unsigned char* mask) {
    const long long ngroups = n / 4;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long g = tid; g < ngroups; g += stride) group<4>(a, g * 4, mask);
    const long long t = ngroups * 4 + tid;
    if (t < n) group<1>(a, t, mask);
}
)K";
    } else if (!P.is_sum) {
        s += R"K(extern "C" __global__ void __launch_bounds__(512) soax_expr_kernel(const Args a, const long long n) {
    const long long ngroups = n / 4;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long g = tid; g < ngroups; g += stride) group<4>(a, g * 4);
    const long long t = ngroups * 4 + tid;
    if (t < n) group<1>(a, t);
}
)K";
    } else {
        // the reduction tree of the hand-written energy kernel (reduce_kernels.cu), restated: per-thread sums in grid-stride
        // order, warp shuffles, one shared-memory step; a fixed grid makes the result run-to-run deterministic
        s += R"K(__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    return x;
}
extern "C" __global__ void __launch_bounds__(256) soax_expr_kernel(const Args a, const long long n, double* partial) {
    __shared__ double sm[32];
    const long long ngroups = n / 4;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    double s = 0.0;
    for (long long g = tid; g < ngroups; g += stride) s += group<4>(a, g * 4);
    const long long t = ngroups * 4 + tid;
    if (t < n) s += group<1>(a, t);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    s = warp_sum(s);
    __syncthreads();
    if (lane == 0) sm[warp] = s;
    __syncthreads();
    if (warp == 0) {
        s = lane < nwarp ? sm[lane] : 0.0;
        s = warp_sum(s);
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}
)K";
    }
    return s;
}

// ---- NVRTC, loaded on first use (the library itself does not link it) ------------------------------------------------------------
struct Nvrtc {
    void* h = nullptr;
    int (*CreateProgram)(void**, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
    int (*CompileProgram)(void*, int, const char* const*) = nullptr;
    int (*GetProgramLogSize)(void*, size_t*) = nullptr;
    int (*GetProgramLog)(void*, char*) = nullptr;
    int (*GetCUBINSize)(void*, size_t*) = nullptr;
    int (*GetCUBIN)(void*, char*) = nullptr;
    int (*DestroyProgram)(void**) = nullptr;
    const char* (*GetErrorString)(int) = nullptr;
    int (*Version)(int*, int*) = nullptr;
    bool wide256 = false;  // PTX ISA 8.8 (CUDA 12.9): ld/st.global.v8.b32
    std::string tried;
};

Nvrtc* nvrtc() {
    static Nvrtc N;
    static std::once_flag once;
    std::call_once(once, [] {
        std::vector<std::string> names;
        if (const char* env = std::getenv("SOAX_NVRTC")) names.push_back(env);
        // absolute toolkit paths first: a bare soname would resolve to whatever NVRTC the process already holds (PyTorch
        // bundles an older one whose PTX ISA lacks the 256-bit accesses)
        for (const char* n : {"/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so", "libnvrtc.so.12", "libnvrtc.so"}) names.push_back(n);
        for (const std::string& n : names) {
            N.h = dlopen(n.c_str(), RTLD_NOW | RTLD_LOCAL);
            if (N.h) break;
            N.tried += n + " ";
        }
        if (!N.h) return;
        auto sym = [&](const char* name) { return dlsym(N.h, name); };
        N.CreateProgram = reinterpret_cast<decltype(N.CreateProgram)>(sym("nvrtcCreateProgram"));
        N.CompileProgram = reinterpret_cast<decltype(N.CompileProgram)>(sym("nvrtcCompileProgram"));
        N.GetProgramLogSize = reinterpret_cast<decltype(N.GetProgramLogSize)>(sym("nvrtcGetProgramLogSize"));
        N.GetProgramLog = reinterpret_cast<decltype(N.GetProgramLog)>(sym("nvrtcGetProgramLog"));
        N.GetCUBINSize = reinterpret_cast<decltype(N.GetCUBINSize)>(sym("nvrtcGetCUBINSize"));
        N.GetCUBIN = reinterpret_cast<decltype(N.GetCUBIN)>(sym("nvrtcGetCUBIN"));
        N.DestroyProgram = reinterpret_cast<decltype(N.DestroyProgram)>(sym("nvrtcDestroyProgram"));
        N.GetErrorString = reinterpret_cast<decltype(N.GetErrorString)>(sym("nvrtcGetErrorString"));
        N.Version = reinterpret_cast<decltype(N.Version)>(sym("nvrtcVersion"));
        int major = 0, minor = 0;
        if (N.Version && N.Version(&major, &minor) == 0) N.wide256 = major > 12 || (major == 12 && minor >= 9);
        if (!N.CreateProgram || !N.CompileProgram || !N.GetCUBINSize || !N.GetCUBIN || !N.DestroyProgram || !N.GetProgramLogSize || !N.GetProgramLog) {
            dlclose(N.h);
            N.h = nullptr;
            N.tried += "(symbols missing) ";
        }
    });
    return N.h ? &N : nullptr;
}

int compile_cubin(const std::string& src, std::vector<char>& cubin) {
    Nvrtc* N = nvrtc();
    if (!N) {
        g_expr_error = "NVRTC is not available (set SOAX_NVRTC to libnvrtc.so.12)";
        return SOAX_ERR_UNSUPPORTED;
    }
    void* prog = nullptr;
    if (N->CreateProgram(&prog, src.c_str(), "soax_expr.cu", 0, nullptr, nullptr) != 0) {
        g_expr_error = "nvrtcCreateProgram failed";
        return SOAX_ERR_ALLOC;
    }
    // the arithmetic contract: no contraction, IEEE division and square root, no flush to zero
    std::vector<const char*> opts = {"--gpu-architecture=sm_100a", "-std=c++17", "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false", "-lineinfo"};
    if (!N->wide256) opts.push_back("-DSOAX_NO_256BIT");  // older NVRTC: a 32-byte access becomes two 128-bit ones
    const int rc = N->CompileProgram(prog, (int)opts.size(), opts.data());
    if (rc != 0) {
        size_t len = 0;
        N->GetProgramLogSize(prog, &len);
        std::string log(len, '\0');
        if (len) N->GetProgramLog(prog, log.data());
        g_expr_error = "NVRTC compilation failed: " + log;
        N->DestroyProgram(&prog);
        return SOAX_ERR_INVALID_ARG;
    }
    size_t len = 0;
    N->GetCUBINSize(prog, &len);
    cubin.resize(len);
    N->GetCUBIN(prog, cubin.data());
    N->DestroyProgram(&prog);
    if (len == 0) {
        g_expr_error = "NVRTC produced no cubin";
        return SOAX_ERR_CUDA;
    }
    return SOAX_OK;
}

}  // namespace

struct CompiledExpr {
    const void* layout_key = nullptr;
    int ncomp = 0, nscalars = 0;
    int bytes_read = 0, bytes_written = 0;
    bool is_sum = false, is_mask = false;
    std::string source, cuda_source;
    std::vector<char> cubin;
    std::mutex mu;
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kernel = nullptr;
};

static bool is_identifier(const char* s) {
    if (!((*s >= 'a' && *s <= 'z') || (*s >= 'A' && *s <= 'Z') || *s == '_')) return false;
    for (; *s; ++s)
        if (!((*s >= 'a' && *s <= 'z') || (*s >= 'A' && *s <= 'Z') || (*s >= '0' && *s <= '9') || *s == '_')) return false;
    return true;
}

static int expr_compile_impl(const ExprLayoutInfo& L, const void* layout_key, const char* source, const char* const* scalar_names,
                             int nscalars, int kind, CompiledExpr** out) {
    const bool is_sum = kind == 1, is_mask = kind == 2;
    g_expr_error.clear();
    Program P;
    P.L = &L;
    for (int k = 0; k < nscalars; ++k) {
        if (!scalar_names[k] || !is_identifier(scalar_names[k])) { g_expr_error = "a scalar name must be an identifier"; return SOAX_ERR_INVALID_ARG; }
        for (int f = 0; f < L.nfields; ++f)
            if (std::strcmp(L.fname[f], scalar_names[k]) == 0) { g_expr_error = std::string("scalar '") + scalar_names[k] + "' has the name of a field"; return SOAX_ERR_INVALID_ARG; }
        P.scalar_names.push_back(scalar_names[k]);
    }
    P.read_first.assign(L.ncomp, false);
    P.assigned.assign(L.ncomp, false);
    P.touched.assign(L.ncomp, false);
    try {
        P.is_sum = is_sum;
        P.is_mask = is_mask;
        Parser parser(source, P);
        if (is_sum) parser.sum_expression();
        else if (is_mask) parser.mask_expression();
        else parser.program();
    } catch (const ParseError& e) {
        char where[64];
        std::snprintf(where, sizeof where, " (at character %zu)", e.pos);
        g_expr_error = e.msg + where;
        return SOAX_ERR_INVALID_ARG;
    }
    bool any = false;
    for (int c = 0; c < L.ncomp; ++c) any |= P.assigned[c];
    if (!any && !is_sum && !is_mask) { g_expr_error = "the program assigns nothing"; return SOAX_ERR_INVALID_ARG; }
    std::unique_ptr<CompiledExpr> E(new (std::nothrow) CompiledExpr());
    if (!E) return SOAX_ERR_ALLOC;
    E->layout_key = layout_key;
    E->ncomp = L.ncomp;
    E->nscalars = nscalars;
    E->is_sum = is_sum;
    E->is_mask = is_mask;
    E->source = source;
    for (int c = 0; c < L.ncomp; ++c) {
        if (P.read_first[c]) E->bytes_read += L.csize[c];
        if (P.assigned[c]) E->bytes_written += L.csize[c];
    }
    if (is_mask) E->bytes_written += 1;
    try {
        E->cuda_source = generate(P);
    } catch (const ParseError& e) {
        g_expr_error = e.msg;
        return SOAX_ERR_INVALID_ARG;
    }
    SOAX_TRY(compile_cubin(E->cuda_source, E->cubin));
    *out = E.release();
    return SOAX_OK;
}

// No C++ exception may cross the C boundary: anything the parser or the standard library throws becomes a status.
int expr_compile(const ExprLayoutInfo& L, const void* layout_key, const char* source, const char* const* scalar_names,
                 int nscalars, int kind, CompiledExpr** out) {
    try {
        return expr_compile_impl(L, layout_key, source, scalar_names, nscalars, kind, out);
    } catch (const std::bad_alloc&) {
        g_expr_error = "out of host memory";
        return SOAX_ERR_ALLOC;
    } catch (...) {
        g_expr_error = "internal error while compiling the program";
        return SOAX_ERR_INVALID_ARG;
    }
}

int expr_run(CompiledExpr* E, const void* layout_key, void* const* comps, int64_t n, const double* scalars, int nscalars,
             cudaStream_t st) {
    if (E->layout_key != layout_key || E->is_sum || E->is_mask) return SOAX_ERR_INVALID_ARG;
    if (nscalars != E->nscalars || (nscalars > 0 && !scalars)) return SOAX_ERR_INVALID_ARG;
    {
        std::lock_guard<std::mutex> lock(E->mu);
        if (!E->kernel) {  // the cubin is loaded into the current context on first use
            SOAX_CUDA(cudaLibraryLoadData(&E->lib, E->cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0));
            SOAX_CUDA(cudaLibraryGetKernel(&E->kernel, E->lib, "soax_expr_kernel"));
        }
    }
    if (n == 0) return SOAX_OK;  // (the code is loaded even then: soax_expr_run relies on it before a stream capture)
    // Args { void* p[ncomp]; double s[max(nscalars,1)]; } -- the layout the generated source declares
    std::vector<unsigned char> args((size_t)E->ncomp * sizeof(void*) + (size_t)(nscalars > 0 ? nscalars : 1) * sizeof(double), 0);
    std::memcpy(args.data(), comps, (size_t)E->ncomp * sizeof(void*));
    if (nscalars > 0) std::memcpy(args.data() + (size_t)E->ncomp * sizeof(void*), scalars, (size_t)nscalars * sizeof(double));
    long long nn = n;
    void* params[] = {args.data(), &nn};
    const int block = g_tune.step_block;
    const int64_t threads = n / 4 > n % 4 ? n / 4 : n % 4;
    const int64_t blocks = (threads + block - 1) / block;
    SOAX_CUDA(cudaLaunchKernel(reinterpret_cast<const void*>(E->kernel), dim3((unsigned)(blocks < 1 ? 1 : blocks)), dim3((unsigned)block), params, 0, st));
    return launched();
}

int sum_partials(const double* partial, int m, double* out, cudaStream_t st);  // reduce_kernels.cu

// A sum program: per-CTA partials from the generated kernel (fixed grid, as the hand-written energy reduction), then the
// library's own fixed-order sum of the partials.
int expr_sum(CompiledExpr* E, const void* layout_key, void* const* comps, int64_t n, const double* scalars, int nscalars,
             double* partial, double* out, cudaStream_t st) {
    if (E->layout_key != layout_key || !E->is_sum) return SOAX_ERR_INVALID_ARG;
    if (nscalars != E->nscalars || (nscalars > 0 && !scalars)) return SOAX_ERR_INVALID_ARG;
    {
        std::lock_guard<std::mutex> lock(E->mu);
        if (!E->kernel) {
            SOAX_CUDA(cudaLibraryLoadData(&E->lib, E->cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0));
            SOAX_CUDA(cudaLibraryGetKernel(&E->kernel, E->lib, "soax_expr_kernel"));
        }
    }
    std::vector<unsigned char> args((size_t)E->ncomp * sizeof(void*) + (size_t)(nscalars > 0 ? nscalars : 1) * sizeof(double), 0);
    std::memcpy(args.data(), comps, (size_t)E->ncomp * sizeof(void*));
    if (nscalars > 0) std::memcpy(args.data() + (size_t)E->ncomp * sizeof(void*), scalars, (size_t)nscalars * sizeof(double));
    long long nn = n;
    void* params[] = {args.data(), &nn, &partial};
    SOAX_CUDA(cudaLaunchKernel(reinterpret_cast<const void*>(E->kernel), dim3(kEnergyBlocks), dim3(256), params, 0, st));
    SOAX_TRY(launched());
    return sum_partials(partial, kEnergyBlocks, out, st);
}

// A mask program: one byte per live particle (1 where the condition holds), same launch shape as expr_run.
int expr_mask(CompiledExpr* E, const void* layout_key, void* const* comps, int64_t n, const double* scalars, int nscalars,
              unsigned char* mask, cudaStream_t st) {
    if (E->layout_key != layout_key || !E->is_mask) return SOAX_ERR_INVALID_ARG;
    if (nscalars != E->nscalars || (nscalars > 0 && !scalars)) return SOAX_ERR_INVALID_ARG;
    {
        std::lock_guard<std::mutex> lock(E->mu);
        if (!E->kernel) {
            SOAX_CUDA(cudaLibraryLoadData(&E->lib, E->cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0));
            SOAX_CUDA(cudaLibraryGetKernel(&E->kernel, E->lib, "soax_expr_kernel"));
        }
    }
    if (n == 0) return SOAX_OK;
    std::vector<unsigned char> args((size_t)E->ncomp * sizeof(void*) + (size_t)(nscalars > 0 ? nscalars : 1) * sizeof(double), 0);
    std::memcpy(args.data(), comps, (size_t)E->ncomp * sizeof(void*));
    if (nscalars > 0) std::memcpy(args.data() + (size_t)E->ncomp * sizeof(void*), scalars, (size_t)nscalars * sizeof(double));
    long long nn = n;
    void* params[] = {args.data(), &nn, &mask};
    const int block = g_tune.step_block;
    const int64_t threads = n / 4 > n % 4 ? n / 4 : n % 4;
    const int64_t blocks = (threads + block - 1) / block;
    SOAX_CUDA(cudaLaunchKernel(reinterpret_cast<const void*>(E->kernel), dim3((unsigned)(blocks < 1 ? 1 : blocks)), dim3((unsigned)block), params, 0, st));
    return launched();
}

void expr_free(CompiledExpr* E) {
    if (!E) return;
    if (E->lib) cudaLibraryUnload(E->lib);
    delete E;
}
const char* expr_error() { return g_expr_error.c_str(); }
const char* expr_cuda_source(const CompiledExpr* E) { return E->cuda_source.c_str(); }
void expr_traffic(const CompiledExpr* E, int* bytes_read, int* bytes_written) {
    if (bytes_read) *bytes_read = E->bytes_read;
    if (bytes_written) *bytes_written = E->bytes_written;
}

}  // namespace soax
