// Test infrastructure: drives the float64 oracle (oracle/oracle_capi.cpp, linked into this executable) under
// AddressSanitizer + UndefinedBehaviorSanitizer.  tests/test_oracle_sanitizers.py builds and runs it; it reads a scenario file
//   n_envs n_drones physics_mode action_type n_steps seed base lo hi n_threads
//   name index value            (one line per parameter entry, passed to orc_params_set)
// resets, steps with the harness action generator, renders every camera's colour frame, and exits 0.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

extern "C" {
void* orc_params_new(int model);
void orc_params_free(void* p);
int orc_params_set(void* p, const char* name, int idx, double value);
void* orc_create(int n_envs, int n_drones, int physics_mode, int action_type, const void* params);
void orc_destroy(void* h);
int orc_obs_dim(const void* h);
void orc_reset(void* h, uint64_t seed);
void orc_step(void* h, const float* actions, int n_threads);
void orc_get_state(const void* h, double* out);
void orc_get_outputs(const void* h, double* obs, double* reward, uint8_t* done, double* margin);
void orc_gen_actions(uint64_t seed, uint32_t t, int n_envs, int n_drones, float base, float lo, float hi, float* out, uint32_t env_base);
void orc_render_rgba(const double* state, int n_envs, int n_drones, const double* cam, double* depth, uint8_t* seg, double* margin,
                     uint8_t* rgba, double* shade, int n_threads);
}

int main(int argc, char** argv) {
    if (argc < 2) return 2;
    FILE* f = std::fopen(argv[1], "r");
    if (!f) return 2;
    int n_envs, n_drones, phys, act, n_steps, n_threads;
    unsigned long long seed;
    float base, lo, hi;
    if (std::fscanf(f, "%d %d %d %d %d %llu %f %f %f %d", &n_envs, &n_drones, &phys, &act, &n_steps, &seed, &base, &lo, &hi, &n_threads) != 10) return 2;
    void* p = orc_params_new(0);
    char name[64];
    int idx;
    double val;
    while (std::fscanf(f, "%63s %d %lf", name, &idx, &val) == 3)
        if (orc_params_set(p, name, idx, val) != 0) { std::fprintf(stderr, "unknown parameter %s[%d]\n", name, idx); return 3; }
    std::fclose(f);
    void* h = orc_create(n_envs, n_drones, phys, act, p);
    if (!h) return 4;
    orc_reset(h, seed);
    const size_t D = (size_t)n_envs * n_drones;
    std::vector<float> a(D * 4);
    std::vector<double> obs((size_t)n_envs * orc_obs_dim(h)), reward(n_envs), margin((size_t)n_envs * 3), state(D * 13);
    std::vector<uint8_t> done(n_envs);
    double sum = 0.0;
    for (int t = 0; t < n_steps; ++t) {
        orc_gen_actions(seed, (uint32_t)t, n_envs, n_drones, base, lo, hi, a.data(), 0u);
        orc_step(h, a.data(), n_threads);
        orc_get_outputs(h, obs.data(), reward.data(), done.data(), margin.data());
        for (double r : reward) sum += r;
    }
    orc_get_state(h, state.data());
    const double cam[10] = {12, 16, 60.0, 0.02, 0.0, 0.0, 0.01, 50.0, 0.0397 + 0.02325, 0.0125};
    const size_t px = 12 * 16;
    std::vector<double> depth(D * px), mg(D * px), shade(D * px);
    std::vector<uint8_t> seg(D * px), rgba(D * px * 4);
    orc_render_rgba(state.data(), n_envs, n_drones, cam, depth.data(), seg.data(), mg.data(), rgba.data(), shade.data(), n_threads);
    unsigned long long chk = 0;
    for (uint8_t v : rgba) chk += v;
    std::printf("ok reward_sum=%.6f rgba_sum=%llu\n", sum, chk);
    orc_destroy(h);
    orc_params_free(p);
    return 0;
}
