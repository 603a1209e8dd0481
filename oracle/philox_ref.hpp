// oracle/philox_ref.hpp — TEST INFRASTRUCTURE (the float64 CPU oracle). Not part of the product:
// only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
// Shares no code with paper_2606_08039_b200/csrc/.
//
// Philox4x32-10 counter-based generator (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy
// as 1, 2, 3", SC'11), restated from the published algorithm; SURVEY.md §8(c) O12 fixes how the
// simulator keys it: key = (seed low 32, seed high 32), counter = (env, drone | 0xFFFFFFFF, control
// step index, stream id).  PAPER.md:254 only says the state "carries a PRNG key"; the counter layout
// is reading Q-O12 in DESIGN.md.
#pragma once
#include <cstdint>

namespace orc {

struct PhiloxOut { uint32_t x[4]; };

inline PhiloxOut philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                               uint32_t k0, uint32_t k1) {
    const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }   // nine key bumps
        const uint64_t prod0 = M0 * (uint64_t)c0;
        const uint64_t prod1 = M1 * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        const uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    PhiloxOut o; o.x[0] = c0; o.x[1] = c1; o.x[2] = c2; o.x[3] = c3;
    return o;
}

// u in [0,1) on a 2^-24 grid: exactly representable in fp32 and fp64.
inline double u01(uint32_t x) { return (double)(x >> 8) * (1.0 / 16777216.0); }

enum : uint32_t { STREAM_RESET_POS = 0, STREAM_RESET_EXTRA = 1, STREAM_WIND = 2, STREAM_ACTION = 3, STREAM_DR0 = 4, STREAM_DR1 = 5, STREAM_DR2 = 6, STREAM_DR3 = 7, STREAM_INIT_RPY = 8, STREAM_INIT_VEL = 9, STREAM_GUST = 10,
                  STREAM_OBS_NOISE = 11 /* 11..13: three calls = 12 normals per drone and step */, STREAM_OBS_BIAS = 14 /* 14..16, per episode */,
                  STREAM_LATENCY = 17 /* per episode: word 0 action latency, word 1 sensor latency */ };
static const uint32_t ENV_LEVEL = 0xFFFFFFFFu;

}  // namespace orc
