// variants.h -- numbering of the per-pair translation variants (celes.h: CELES_TRANSLATION_*).
#pragma once

// How W^{ii'} b^{i'} is evaluated per pair (celes.h: CELES_TRANSLATION_*)
namespace celes {
constexpr int kRotated = 0;         // packed FFMA2 rotate / axial-translate / rotate (default)
constexpr int kDirect = 1;          // term-by-term sum of (A.6)-(A.8), the paper's algorithm
}  // namespace celes
