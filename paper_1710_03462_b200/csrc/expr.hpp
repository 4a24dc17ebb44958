// expr.hpp -- interface between the C ABI (api.cu) and the expression compiler (expr.cu).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "layout.hpp"

namespace soax {

// What the expression compiler needs to know about a layout: names, dimensions and component types.
struct ExprLayoutInfo {
    int nfields, ncomp;
    const char* fname[kMaxComp];
    int fdim[kMaxComp], fbegin[kMaxComp];
    int cdtype[kMaxComp], csize[kMaxComp];
};

struct CompiledExpr;
// kind: 0 = assignment program (expr_run), 1 = sum of one expression (expr_sum), 2 = mask of one condition (expr_mask)
int expr_compile(const ExprLayoutInfo& L, const void* layout_key, const char* source, const char* const* scalar_names,
                 int nscalars, int kind, CompiledExpr** out);
int expr_run(CompiledExpr* e, const void* layout_key, void* const* comps, int64_t n, const double* scalars, int nscalars,
             cudaStream_t st);
int expr_sum(CompiledExpr* e, const void* layout_key, void* const* comps, int64_t n, const double* scalars, int nscalars,
             double* partial, double* out, cudaStream_t st);
int expr_mask(CompiledExpr* e, const void* layout_key, void* const* comps, int64_t n, const double* scalars, int nscalars,
              unsigned char* mask, cudaStream_t st);
void expr_free(CompiledExpr* e);
const char* expr_error();
const char* expr_cuda_source(const CompiledExpr* e);
void expr_traffic(const CompiledExpr* e, int* bytes_read, int* bytes_written);

}  // namespace soax
