// Test infrastructure: builds plans for many topologies and option sets with csrc/plan.cpp compiled under
// -fsanitize=address,undefined (tests/test_plan_sanitizers.py).  Host only; the device side is stubbed out.
#include <cstdio>
#include <cstdlib>
#include <vector>
#include <string>
#include "plan_internal.h"
namespace hines { struct DeviceTables {}; }
extern "C" hines_status_t hines_plan_destroy(hines_plan_t* P) { delete P; return HINES_OK; }
template <typename T> static std::vector<T> rd(const std::string& f) { FILE* fp = fopen(f.c_str(), "rb"); fseek(fp, 0, SEEK_END); long n = ftell(fp); fseek(fp, 0, SEEK_SET); std::vector<T> v(n / sizeof(T)); if (fread(v.data(), 1, n, fp) != (size_t)n) abort(); fclose(fp); return v; }
int main(int argc, char** argv) {
    int ncase = atoi(argv[1]);
    struct O { int flags, seg, chunk, clmax, smem, split, dtype; };
    O opts[] = {{0,0,0,0,0,0,0}, {0,0,0,0,0,0,1}, {2,0,0,0,0,0,0}, {128,0,0,0,0,0,0}, {512,0,0,0,0,0,0}, {0,7,30000,16,0,0,0}, {0,9,0,2,64000,12000,0}, {8,0,0,0,60000,0,0}, {1,0,0,0,0,0,0}, {256,3,0,0,0,0,1}, {4,0,0,0,0,0,0}, {64,0,20000,2,48000,20000,0}, {4096,0,0,0,0,0,0}, {4096,0,20000,2,48000,20000,0}};
    long plans = 0;
    for (int k = 0; k < ncase; ++k) {
        auto par = rd<int32_t>(std::string(argv[2]) + "/p" + std::to_string(k) + ".bin"); auto offs = rd<int64_t>(std::string(argv[2]) + "/o" + std::to_string(k) + ".bin");
        for (const O& o : opts) {
            hines_options_t op{}; op.struct_size = sizeof(op); op.policy_flags = o.flags; op.max_segment = o.seg; op.chunk_smem_bytes = o.chunk; op.cluster_max = o.clmax; op.smem_bytes_per_block = o.smem; op.split_smem_bytes = o.split;
            hines_plan_t* P = nullptr;
            hines_status_t st = hines_plan_create(par.data(), offs.data(), (int64_t)offs.size() - 1, (hines_dtype_t)o.dtype, &op, &P);
            if (st != HINES_OK) { printf("case %d flags %d: %s (%s)\n", k, o.flags, hines_status_string(st), hines_last_error()); continue; }
            hines_plan_info_t info; hines_plan_get_info(P, &info);
            std::vector<int32_t> part(offs.size() - 1); std::vector<int64_t> cost(3);
            hines_partition_cells(offs.data(), (int64_t)offs.size() - 1, 3, part.data(), cost.data());
            ++plans; hines_plan_destroy(P);
        }
    }
    printf("plans built under ASan/UBSan: %ld\n", plans);
    return 0;
}
