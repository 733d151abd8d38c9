// tables.cu -- host-side FP64 table builder, plan caches, error string, launch accounting.
//
// Tables follow DESIGN.md readings R1/R2/R8/R9: orthonormal real spherical harmonics without
// Condon-Shortley phase (PAPER.md:663 Eq.(C1)), Gauss-Legendre nodes in x = cos(theta) with weights
// summing to 2, phi_v = 2 pi v / V, inverse transform weight 2 pi / V (Eq.(39) :339).
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace cgtp {

// ------------------------------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}
void clear_error() { g_err[0] = 0; }
const char* last_error() { return g_err; }

// ------------------------------------------------------------------- per-device facts, path switch
static std::mutex g_dev_mu;
static int g_sms[64] = {0};
int num_sms()
{
    const int dev = current_device();
    if (dev < 0 || dev >= 64) return 148;
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (!g_sms[dev]) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        g_sms[dev] = n;
    }
    return g_sms[dev];
}

static thread_local bool g_pdl_plain = false;
bool pdl_plain() { return g_pdl_plain; }
void set_pdl_plain(bool plain) { g_pdl_plain = plain; }

static int g_kernel_path = 0;
int kernel_path() { return g_kernel_path; }
void set_kernel_path(int flags) { g_kernel_path = flags; }

// --------------------------------------------------------------------------- launch accounting
static std::mutex g_prof_mu;
static int64_t g_launches = 0;
static bool g_prof_on = false;
struct ProfRec {
    Kind kind;
    cudaEvent_t e0, e1;
};
static std::vector<ProfRec*> g_recs;

LaunchScope::LaunchScope(Kind k, cudaStream_t s) : kind(k), stream(s), rec(nullptr)
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    ++g_launches;
    if (g_prof_on) {
        ProfRec* r = new ProfRec;
        r->kind = k;
        cudaEventCreate(&r->e0);
        cudaEventCreate(&r->e1);
        cudaEventRecord(r->e0, s);
        rec = r;
    }
}
LaunchScope::~LaunchScope()
{
    if (rec) {
        ProfRec* r = static_cast<ProfRec*>(rec);
        cudaEventRecord(r->e1, stream);
        std::lock_guard<std::mutex> lk(g_prof_mu);
        g_recs.push_back(r);
    }
}

int64_t launch_count()
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    return g_launches;
}
void profile_enable(bool on)
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_on = on;
}
int profile_collect(double* ms, int64_t* launches)
{
    std::vector<ProfRec*> recs;
    {
        std::lock_guard<std::mutex> lk(g_prof_mu);
        recs.swap(g_recs);
    }
    int rc = CGTP_OK;
    for (ProfRec* r : recs) {
        float t = 0.f;
        cudaError_t e = cudaEventSynchronize(r->e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, r->e0, r->e1);
        if (e != cudaSuccess) {
            set_error("profile_collect: %s", cudaGetErrorString(e));
            rc = CGTP_ERR_CUDA;
        } else {
            if (ms) ms[r->kind] += t;
            if (launches) launches[r->kind] += 1;
        }
        cudaEventDestroy(r->e0);
        cudaEventDestroy(r->e1);
        delete r;
    }
    return rc;
}

// ------------------------------------------------------------------------------ Gauss-Legendre
// Nodes by Newton iteration on P_U, northern node first; exact mirror symmetry is enforced.
void gauss_legendre(int U, std::vector<double>& x, std::vector<double>& w)
{
    x.assign(U, 0.0);
    w.assign(U, 0.0);
    for (int i = 0; i < (U + 1) / 2; ++i) {
        double z = std::cos(M_PI * (i + 0.75) / (U + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = z;
            for (int k = 2; k <= U; ++k) {
                double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            dp = U * (z * p1 - p0) / (z * z - 1.0);
            double dz = p1 / dp;
            z -= dz;
            if (std::fabs(dz) < 1e-16) break;
        }
        {
            double p0 = 1.0, p1 = z;
            for (int k = 2; k <= U; ++k) {
                double p2 = ((2.0 * k - 1.0) * z * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            dp = U * (z * p1 - p0) / (z * z - 1.0);
        }
        x[i] = z;
        x[U - 1 - i] = -z;
        w[i] = w[U - 1 - i] = 2.0 / ((1.0 - z * z) * dp * dp);
    }
    if (U % 2) x[U / 2] = 0.0;
}

// P[u][l][m] = P~_l^m(x_u), 0 <= m <= l <= LB: orthonormal on S^2 (R1), no Condon-Shortley phase (R2).
void legendre_values(int U, int LB, const std::vector<double>& x, std::vector<double>& P)
{
    const int LL = LB + 1;
    P.assign((size_t)U * LL * LL, 0.0);
    auto at = [&](int u, int l, int m) -> double& { return P[((size_t)u * LL + l) * LL + m]; };
    for (int u = 0; u < U; ++u) {
        double ct = x[u], st = std::sqrt(1.0 - ct * ct);
        at(u, 0, 0) = std::sqrt(1.0 / (4.0 * M_PI));
        for (int m = 1; m <= LB; ++m) at(u, m, m) = std::sqrt((2.0 * m + 1.0) / (2.0 * m)) * st * at(u, m - 1, m - 1);
        for (int m = 0; m <= LB; ++m) {
            if (m + 1 <= LB) at(u, m + 1, m) = std::sqrt(2.0 * m + 3.0) * ct * at(u, m, m);
            for (int l = m + 2; l <= LB; ++l) {
                double a = std::sqrt((4.0 * l * l - 1.0) / ((double)l * l - (double)m * m));
                double b = std::sqrt(((l - 1.0) * (l - 1.0) - (double)m * m) / (4.0 * (l - 1.0) * (l - 1.0) - 1.0));
                at(u, l, m) = a * (ct * at(u, l - 1, m) - b * at(u, l - 2, m));
            }
        }
    }
}

// ------------------------------------------------------------------------------------ plan cache
static std::mutex g_plan_mu;
static std::vector<Plan*> g_plans;

static const float* upload(const std::vector<float>& h, bool* ok)
{
    float* d = nullptr;
    size_t bytes = h.size() * sizeof(float);
    if (cudaMalloc(&d, bytes) != cudaSuccess) { *ok = false; return nullptr; }
    if (cudaMemcpy(d, h.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) { *ok = false; return nullptr; }
    return d;
}

const Plan* get_plan(int lmax, int lmax_out) { return get_plan_nu(lmax, lmax_out, 2); }

const Plan* get_plan_nu(int lmax, int lmax_out, int nu)
{
    const int dev = current_device();
    std::lock_guard<std::mutex> lk(g_plan_mu);
    for (Plan* p : g_plans)
        if (p->dev == dev && p->lmax == lmax && p->lmax_out == lmax_out && p->nu == nu) return p;

    Plan* p = new Plan;
    std::memset(p, 0, sizeof *p);
    p->dev = dev;
    p->lmax = lmax;
    p->lmax_out = lmax_out;
    p->nu = nu;
    const int LB = p->LB = kernel_band(lmax > lmax_out ? lmax : lmax_out);
    // a product of nu fields of band lmax against Y_lm, l <= lmax_out, is a polynomial of degree nu lmax + lmax_out
    const int U = p->U = (nu * lmax + lmax_out + 2) / 2;  // ceil((nu lmax + lmax_out + 1)/2)
    const int V = p->V = nu * lmax + lmax_out + 1;
    const int Uh = p->Uh = (U + 1) / 2;
    const int Vh = p->Vh = V / 2 + 1;
    p->UV = U * V;
    p->UVp = round_up(U * V, 4);
    const int NTRI = p->NTRI = round_up((LB + 1) * (LB + 2) / 2, 4);
    const int QSTR = p->QSTR = round_up(LB + 1, 4);
    p->L2 = (lmax + 1) * (lmax + 1);
    p->L2p = round_up(p->L2, 4);
    p->Lo2 = (lmax_out + 1) * (lmax_out + 1);
    p->Lo2p = round_up(p->Lo2, 4);

    std::vector<double> x, w;
    gauss_legendre(U, x, w);

    // normalised associated Legendre functions at every node (FP64), P[u][l][m]
    const int LL = LB + 1;
    std::vector<double> P;
    legendre_values(U, LB, x, P);
    auto at = [&](int u, int l, int m) -> double& { return P[((size_t)u * LL + l) * LL + m]; };

    std::vector<float> PT((size_t)Uh * NTRI, 0.f), DT(PT), ST(PT), WP(PT), WD(PT), WS(PT);
    for (int u = 0; u < Uh; ++u) {
        double ct = x[u], st = std::sqrt(1.0 - ct * ct);
        double wu = w[u] * ((U % 2 && u == Uh - 1) ? 0.5 : 1.0);
        for (int l = 0; l <= LB; ++l)
            for (int m = 0; m <= l; ++m) {
                double pv = at(u, l, m);
                double pm1 = (l - 1 >= m) ? at(u, l - 1, m) : 0.0;
                // d/dtheta P~_l^m = (l x P~_l^m - sqrt((2l+1)(l^2-m^2)/(2l-1)) P~_{l-1}^m) / sin(theta)
                double c = (l > 0) ? std::sqrt((2.0 * l + 1.0) * ((double)l * l - (double)m * m) / (2.0 * l - 1.0)) : 0.0;
                double dth = (l * ct * pv - c * pm1) / st;
                size_t k = (size_t)u * NTRI + tri_index(l, m);
                PT[k] = (float)pv;
                DT[k] = (float)dth;
                ST[k] = (float)(m * pv / st);
                WP[k] = (float)(wu * pv);
                WD[k] = (float)(wu * dth);
                WS[k] = (float)(wu * m * pv / st);
            }
    }

    std::vector<float> QC((size_t)Vh * QSTR, 0.f), QS(QC), WV(round_up(Vh, 4), 0.f);
    for (int v = 0; v < Vh; ++v) {
        double ph = 2.0 * M_PI * v / V;
        bool paired = (v != 0) && !(V % 2 == 0 && v == V / 2);
        WV[v] = (float)((2.0 * M_PI / V) * (paired ? 1.0 : 0.5));
        for (int m = 0; m <= LB; ++m) {
            QC[(size_t)v * QSTR + m] = (float)(m == 0 ? 1.0 : std::sqrt(2.0) * std::cos(m * ph));
            QS[(size_t)v * QSTR + m] = (float)((m == 0 || !paired) ? 0.0 : std::sqrt(2.0) * std::sin(m * ph));
        }
    }

    std::vector<float> geo((size_t)8 * p->UVp, 0.f);
    for (int u = 0; u < U; ++u) {
        double ct = x[u], st = std::sqrt(1.0 - ct * ct);
        for (int v = 0; v < V; ++v) {
            double ph = 2.0 * M_PI * v / V, cp = std::cos(ph), sp = std::sin(ph);
            size_t q = (size_t)u * V + v;
            geo[0 * p->UVp + q] = (float)(st * cp);
            geo[1 * p->UVp + q] = (float)(st * sp);
            geo[2 * p->UVp + q] = (float)ct;
            geo[3 * p->UVp + q] = (float)(ct * cp);
            geo[4 * p->UVp + q] = (float)(ct * sp);
            geo[5 * p->UVp + q] = (float)(-st);
            geo[6 * p->UVp + q] = (float)(-sp);
            geo[7 * p->UVp + q] = (float)cp;
        }
    }

    bool ok = true;
    p->PT = upload(PT, &ok);
    p->DT = upload(DT, &ok);
    p->ST = upload(ST, &ok);
    p->WP = upload(WP, &ok);
    p->WD = upload(WD, &ok);
    p->WS = upload(WS, &ok);
    p->QC = upload(QC, &ok);
    p->QS = upload(QS, &ok);
    p->WV = upload(WV, &ok);
    p->geo = upload(geo, &ok);
    if (!ok) {
        set_error("get_plan(%d,%d): device table upload failed: %s", lmax, lmax_out,
                  cudaGetErrorString(cudaGetLastError()));
        delete p;
        return nullptr;
    }
    auto keep = [](const std::vector<float>& v) {
        float* h = new float[v.size()];
        std::memcpy(h, v.data(), v.size() * sizeof(float));
        return h;
    };
    p->hQC = keep(QC);
    p->hQS = keep(QS);
    p->hWV = keep(WV);
    g_plans.push_back(p);
    return p;
}

// ---------------------------------------------------------------------------- channel plan cache
static std::mutex g_chan_mu;
struct ChanEntry {
    ChannelPlan plan;
    std::vector<uint8_t> mask;
};
static std::vector<ChanEntry*> g_chans;

const ChannelPlan* get_channel_plan(int C, const uint8_t* mask)
{
    const int dev = current_device();
    std::lock_guard<std::mutex> lk(g_chan_mu);
    for (ChanEntry* e : g_chans)
        if (e->plan.dev == dev && e->plan.C == C && std::memcmp(e->mask.data(), mask, C) == 0) return &e->plan;
    ChanEntry* e = new ChanEntry;
    e->mask.assign(mask, mask + C);
    e->plan.dev = dev;
    e->plan.C = C;
    int k = 0;
    for (int c = 0; c < C; ++c)
        if (mask[c] == 0) e->plan.perm_host[k++] = c;
    e->plan.Ce = k;
    for (int c = 0; c < C; ++c)
        if (mask[c] != 0) e->plan.perm_host[k++] = c;
    e->plan.Co = C - e->plan.Ce;
    int* d = nullptr;
    if (cudaMalloc(&d, sizeof(int) * C) != cudaSuccess ||
        cudaMemcpy(d, e->plan.perm_host, sizeof(int) * C, cudaMemcpyHostToDevice) != cudaSuccess) {
        set_error("get_channel_plan: device upload failed: %s", cudaGetErrorString(cudaGetLastError()));
        delete e;
        return nullptr;
    }
    e->plan.perm_dev = d;
    g_chans.push_back(e);
    return &e->plan;
}

}  // namespace cgtp
