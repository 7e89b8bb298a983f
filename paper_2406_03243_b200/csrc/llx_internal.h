// Shared by the translation units of libllx.so (not part of the ABI).
#pragma once
#include <new>

#include "../../include/llx.h"

namespace llx {
// Records the thread's llx_last_error() text and returns `s`.
llx_status fail(llx_status s, const char* fmt, ...);
}  // namespace llx

// llx.h: "nothing throws or aborts across this boundary".  Entry points that allocate host memory (std::vector,
// unordered_map) run between these two: an allocation failure becomes LLX_ERR_OOM.
#define LLX_TRY try {
#define LLX_CATCH                                                                     \
    }                                                                                 \
    catch (const std::bad_alloc&) { return llx::fail(LLX_ERR_OOM, "host allocation failed"); } \
    catch (...) { return llx::fail(LLX_ERR_INVALID_ARG, "unexpected C++ exception"); }
