// lm_specs.cuh -- chain structures that get an ahead-of-time specialised kernel.
//
// A ChainSpec fixes only the STRUCTURE of a modified-DH table (joint types, which twists are 0 or
// +-pi/2, which offsets are exactly zero); the non-zero lengths stay run-time data in KChain.  At
// lm_init the structure of the caller's chain is computed (lm_api.cu: chain_signature) and compared
// with every entry below; a match selects the specialised kernel, anything else runs the generic
// one (same results: the specialisation only removes multiplications by exact 0 / +-1).
#pragma once
#include "lm_device.cuh"

namespace lmk {

// Franka Panda (BASELINE.json configs[0,1,3,4]): 7 revolute joints,
//   alpha = (0, -, +, +, -, +, +) * pi/2,  a != 0 at joints 4, 5, 7,  d != 0 at joints 1, 3, 5,
//   no theta offsets, flange = pure z translation.
struct PandaSpec {
    static constexpr ChainSpec spec = {false, 7, /*pris*/ 0x00, /*al0*/ 0x01, /*alp*/ 0x6C, /*aln*/ 0x12,
                                       /*a0*/ 0x27, /*d0*/ 0x6A, /*t0*/ 0x7F, /*tool_rot*/ false, /*tp0*/ 0x3};
};

// The seeded random 8-DoF chain of BASELINE.json configs[2] (workloads.random_chain_8dof(3)):
// joint 1 prismatic, alpha = (0, -, +, 0, -, -, -, 0) * pi/2, a != 0 at joints 2-5 and 8,
// d != 0 at joints 6, 7, theta offsets on every revolute joint, tool = pure z translation.
struct Rand8Spec {
    static constexpr ChainSpec spec = {false, 8, /*pris*/ 0x01, /*al0*/ 0x89, /*alp*/ 0x04, /*aln*/ 0x72,
                                       /*a0*/ 0x61, /*d0*/ 0x9F, /*t0*/ 0x01, /*tool_rot*/ false, /*tp0*/ 0x3};
};

enum SpecId : int { SPEC_GENERIC = 0, SPEC_PANDA = 1, SPEC_RAND8 = 2, SPEC_COUNT = 3 };

inline const ChainSpec *registered_spec(int id) {
    static const ChainSpec panda = PandaSpec::spec, rand8 = Rand8Spec::spec;
    return id == SPEC_PANDA ? &panda : id == SPEC_RAND8 ? &rand8 : nullptr;
}
inline const char *spec_name(int id) { return id == SPEC_PANDA ? "panda7" : id == SPEC_RAND8 ? "rand8" : "generic"; }

} // namespace lmk
