// Shared by the translation units of libllx.so (not part of the ABI).
#pragma once
#include "../../include/llx.h"

namespace llx {
// Records the thread's llx_last_error() text and returns `s`.
llx_status fail(llx_status s, const char* fmt, ...);
}  // namespace llx
