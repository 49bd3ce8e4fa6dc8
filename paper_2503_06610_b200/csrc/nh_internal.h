// nh_internal.h -- what the library's translation units share on the host side (nothing of the method).
#pragma once

namespace nh {
// Store `msg` as the calling thread's nh_last_error() text and return `code` (defined in nh_api.cu).
int set_error(int code, const char* msg);
}  // namespace nh
