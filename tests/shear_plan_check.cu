// shear_plan_check.cu — runs the HOST plan of the sheared-plane kernel (make_shear_plan of vr_shear.cu) on given
// cameras and replays, per beam, the decisions the kernel prologue takes with the same geometry functions: would
// the beam fit its plane slots (else it marches through global memory — correct but slow, a tail), and does every
// plane the planner would stage fit (else the overflow flag).  Host code only (nvcc, no GPU); input = lines of
// "nx ny nz W H step" + 18 camera floats, written by tests/test_shear_plan.py from workload/.  Test infrastructure.
#include <cstdarg>
#include <cstdio>
#include <cstdlib>

#include "../paper_1111_6661_b200/csrc/vr_shear.cu"

namespace vr {                       // the two symbols vr_shear.cu takes from vr_api.cu
void set_error(const char *, ...) {}
vr_status cuda_fail(cudaError_t, const char *) { return VR_ERR_CUDA; }
}

using namespace vr;

// C.1 / C.2 / C.3 in float32 with correctly rounded fmaf, as vr_math.cuh does on the device
struct HRay { float d[3], oc[3], t_first, t_exit; bool hit; };
static HRay host_ray(const CamK &c, const int n[3], int i, int j)
{
    HRay r;
    const float px = (float)i + 0.5f, py = (float)j + 0.5f;
    float o[3], g[3];
    for (int a = 0; a < 3; ++a) {
        o[a] = fmaf(py, c.ov[a], fmaf(px, c.ou[a], c.o0[a]));
        g[a] = fmaf(py, c.dv[a], fmaf(px, c.du[a], c.d0[a]));
    }
    const float len = sqrtf(fmaf(g[2], g[2], fmaf(g[1], g[1], g[0] * g[0])));
    float t_enter = 0.0f, t_exit = INFINITY;
    r.hit = true;
    for (int a = 0; a < 3; ++a) {
        r.d[a] = g[a] / len;
        float lo = -INFINITY, hi = INFINITY;
        if (r.d[a] != 0.0f) {
            const float inv = 1.0f / r.d[a];
            const float ta = (0.0f - o[a]) * inv, tb = ((float)n[a] - o[a]) * inv;
            lo = fminf(ta, tb); hi = fmaxf(ta, tb);
        } else if (o[a] < 0.0f || o[a] > (float)n[a]) r.hit = false;
        t_enter = fmaxf(t_enter, lo); t_exit = fminf(t_exit, hi);
        r.oc[a] = o[a] - 0.5f;
    }
    if (!(t_exit > t_enter)) r.hit = false;
    r.t_first = fmaf(0.5f, c.step, t_enter); r.t_exit = t_exit;
    return r;
}
static int host_cell(float t, float d, float oc, int n)
{
    float q = fmaf(t, d, oc);
    q = fminf(fmaxf(q, 0.0f), (float)(n - 1));
    return std::min((int)floorf(q), n - 2);
}

int main(int argc, char **argv)
{
    if (argc < 2) return 2;
    FILE *f = fopen(argv[1], "r");
    if (!f) return 2;
    long long tot_direct = 0, tot_overflow = 0, tot_beams = 0;
    int view = 0;
    for (;; ++view) {
        int n[3], W, H;
        float step, v[18];
        if (fscanf(f, "%d %d %d %d %d %f", &n[0], &n[1], &n[2], &W, &H, &step) != 6) break;
        for (int k = 0; k < 18; ++k) if (fscanf(f, "%f", &v[k]) != 1) return 2;
        CamK cam;
        for (int a = 0; a < 3; ++a) {
            cam.o0[a] = v[a]; cam.ou[a] = v[3 + a]; cam.ov[a] = v[6 + a];
            cam.d0[a] = v[9 + a]; cam.du[a] = v[12 + a]; cam.dv[a] = v[15 + a];
        }
        cam.step = step; cam.t_min = 0.01f; cam.width = W; cam.height = H;
        ShearPlanK P;
        unsigned int smem = 0;
        const bool fits = make_shear_plan(false, cam, n, nullptr, P, smem);
        long long beams = 0, direct_fit = 0, direct_oblique = 0, overflow = 0;
        double staged = 0.0;                        // bytes the frame copies into shared memory
        for (int ty = 0; fits && ty * kBH < H; ++ty)
            for (int tx = 0; tx * kBW < W; ++tx) {
                const int x0 = tx * kBW, y0 = ty * kBH;
                float oc[3], gc[3];
                cam_ray_at(cam, (float)x0 + 0.5f * kBW, (float)y0 + 0.5f * kBH, oc, gc);
                const int a = principal_axis(gc), sgn = gc[a] > 0.0f ? 1 : -1;
                int au, av;
                beam_axes(a, au, av);
                int iw_min = INT_MAX, iw_max = INT_MIN;
                for (int j = y0; j < std::min(y0 + kBH, H); ++j)
                    for (int i = x0; i < std::min(x0 + kBW, W); ++i) {
                        const HRay r = host_ray(cam, n, i, j);
                        if (!r.hit || !(r.t_first < r.t_exit)) continue;
                        const int ia = host_cell(r.t_first, r.d[a], r.oc[a], n[a]), ib = host_cell(r.t_exit, r.d[a], r.oc[a], n[a]);
                        iw_min = std::min(iw_min, std::min(ia, ib)); iw_max = std::max(iw_max, std::max(ia, ib));
                    }
                if (iw_min > iw_max) continue;                 // the whole beam misses
                ++beams;
                BeamLine L[4];
                bool ok = true;
                for (int k = 0; k < 4 && ok; ++k)
                    ok = beam_line(cam, (float)((k & 1) ? std::min(x0 + kBW, W) : x0), (float)((k & 2) ? std::min(y0 + kBH, H) : y0), a, sgn, L[k]);
                if (!ok) { ++direct_oblique; continue; }
                int wb, hb;
                beam_rect_bound(L, iw_min, iw_max + 1, n[a], n[au], n[av], wb, hb);
                if (!(std::min(wb + 1, n[au]) <= P.PU[a] && std::min(hb + 1, n[av]) <= P.PV[a])) { ++direct_fit; continue; }
                for (int q = iw_min; q <= iw_max + 1; ++q) {
                    int u0, v0, w, h;
                    plane_rect(L, q, n[a], n[au], n[av], false, u0, v0, w, h);
                    if (w > P.PU[a] || h > P.PV[a]) ++overflow;
                    staged += 4.0 * w * h;
                }
            }
        const int ctas = std::min(3, (int)(kSmemSM / (smem + 1024u)));
        printf("view %d: %dx%dx%d %dx%d fits %d smem %u ctas %d | x: PU %d PV %d G %d | y: PU %d PV %d G %d | z: PU %d PV %d G %d | beams %lld direct_fit %lld direct_oblique %lld overflow %lld staged %.2f GB = %.2f x volume\n",
               view, n[0], n[1], n[2], W, H, (int)fits, smem, ctas, P.PU[0], P.PV[0], P.G[0], P.PU[1], P.PV[1], P.G[1], P.PU[2], P.PV[2], P.G[2],
               beams, direct_fit, direct_oblique, overflow, staged / 1e9, staged / (4.0 * n[0] * n[1] * n[2]));
        for (int a = 0; a < 3 && fits; ++a)
            if (P.NS[a] < 2 * P.G[a] + 1 || P.G[a] + 1 > kMaxLoad || 3 * P.G[a] + 1 > 64 || P.PP[a] < P.PU[a] * P.PV[a] || smem > kSmemMax) ++overflow;
        tot_direct += direct_fit; tot_overflow += overflow; tot_beams += beams;
    }
    fclose(f);
    printf("total beams %lld direct_fit %lld overflow %lld\n", tot_beams, tot_direct, tot_overflow);
    return (tot_direct || tot_overflow || tot_beams == 0) ? 1 : 0;
}
