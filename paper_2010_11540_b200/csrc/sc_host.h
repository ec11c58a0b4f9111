// sc_host.h -- host-side declarations shared by the library's translation units (product code only).
#pragma once
#include <string>

namespace sc {
// Store the message sc_last_error(NULL) returns on this thread (calls that have no context to keep it in).
void set_global_error(const std::string& msg);
}  // namespace sc
