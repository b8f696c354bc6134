// Device math helpers of the PIMD hot path: exp for the log-sum-exp passes and the Gaussian pair
// kernel, double-double differences, signed log-sum-exp accumulators, Philox4x32-10.
// Nothing here is shared with oracle/ (the oracle has its own plain-C versions).
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#define PIMD_DEV __device__ __forceinline__

namespace pimd {

// ---------------------------------------------------------------------------------------------
// exp(x) for x <= ~700, no special-case branches: 0 for x < -708 (and for -inf), garbage-in /
// garbage-out for NaN (non-finite state is detected elsewhere).  Cody-Waite reduction
// x = k ln2 + r, |r| <= ln2/2, degree-13 Taylor polynomial (truncation 4e-18), 2^k folded into
// the exponent field.  17 FP64 instructions; max relative error ~2e-16.
// ---------------------------------------------------------------------------------------------
PIMD_DEV double exp_fast(double x)
{
    const double MAGIC = 6755399441055744.0; // 1.5 * 2^52
    double t = fma(x, 1.4426950408889634074, MAGIC);
    int k = __double2loint(t);
    double kd = t - MAGIC;
    double r = fma(kd, -6.93147180369123816490e-01, x);
    r = fma(kd, -1.90821492927058770002e-10, r);
    double p = 1.6059043836821613e-10;           // 1/13!
    p = fma(p, r, 2.08767569878680989792e-09);   // 1/12!
    p = fma(p, r, 2.50521083854417187751e-08);   // 1/11!
    p = fma(p, r, 2.75573192239858906526e-07);   // 1/10!
    p = fma(p, r, 2.75573192239858906526e-06);   // 1/9!
    p = fma(p, r, 2.48015873015873015873e-05);   // 1/8!
    p = fma(p, r, 1.98412698412698412698e-04);   // 1/7!
    p = fma(p, r, 1.38888888888888888889e-03);   // 1/6!
    p = fma(p, r, 8.33333333333333333333e-03);   // 1/5!
    p = fma(p, r, 4.16666666666666666667e-02);   // 1/4!
    p = fma(p, r, 1.66666666666666666667e-01);   // 1/3!
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    int hi = __double2hiint(p) + (k << 20);
    double res = __hiloint2double(hi, __double2loint(p));
    return (x < -708.0) ? 0.0 : res;
}

// ---------------------------------------------------------------------------------------------
// exp(x) for x <= 0 (the Gaussian pair factor), table driven: x = j ln2/32 + r, |r| <= ln2/64,
// exp(x) = 2^(j>>5) * 2^((j&31)/32) * P6(r); degree-6 Taylor remainder 3.5e-18.  11 FP64
// instructions + one shared-memory lookup; max relative error ~3e-16.  0 for x < -708.
// `tab` points to the 32 doubles 2^(i/32) in shared memory (copied from c_exp2_32).
// ---------------------------------------------------------------------------------------------
__constant__ double c_exp2_32[32] = {
    1.0, 1.0218971486541166, 1.0442737824274138, 1.0671404006768237,
    1.0905077326652577, 1.1143867425958924, 1.1387886347566916, 1.1637248587775775,
    1.189207115002721, 1.215247359980469, 1.241857812073484, 1.2690509571917332,
    1.2968395546510096, 1.3252366431597413, 1.3542555469368927, 1.383909881963832,
    1.4142135623730951, 1.4451808069770467, 1.4768261459394993, 1.5091644275934228,
    1.5422108254079407, 1.5759808451078865, 1.6104903319492543, 1.645755478153965,
    1.681792830507429, 1.718619298122478, 1.7562521603732995, 1.7947090750031072,
    1.8340080864093424, 1.8741676341103, 1.9152065613971474, 1.9571441241754002};

PIMD_DEV double exp_tab(double x, const double *tab)
{
    const double MAGIC = 6755399441055744.0; // 1.5 * 2^52
    const double t = fma(x, 46.16624130844683, MAGIC); // 32 / ln 2
    const int j = __double2loint(t);
    const double kd = t - MAGIC;
    double r = fma(kd, -0.02166084938653512, x);       // ln2/32, upper 33 bits (kd * hi is exact)
    r = fma(kd, -5.9631716539705866e-12, r);
    double p = 1.0 / 720.0;
    p = fma(p, r, 1.0 / 120.0);
    p = fma(p, r, 1.0 / 24.0);
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    const double v = tab[j & 31] * p;
    const bool uf = (unsigned)__double2hiint(x) > 0xC0862000u; // x < -708 (or NaN): integer compare, off the FP64 pipe
    const int hi = __double2hiint(v) + ((j >> 5) << 20);
    return __hiloint2double(uf ? 0 : hi, uf ? 0 : __double2loint(v));
}

// ---------------------------------------------------------------------------------------------
// exp(-r2) for r2 >= 0 (the Gaussian pair factor), 64-entry table: -r2 = j ln2/64 + r, |r| <= ln2/128,
// exp(-r2) = 2^(j>>6) * 2^((j&63)/64) * P5(r); degree-5 Taylor remainder 3.5e-17.  9 FP64
// instructions, no FP64 compare: r2 is clamped to 708 through its high word (integer min), so the
// smallest value returned is e^-708 = 3e-308 instead of 0.  One FMA reduction: the rounding of ln2/64
// costs a relative error r2 * 1.1e-16, i.e. at most 4e-17 of the largest term.
// `tab` points to the 64 doubles 2^(i/64) in shared memory (copied from c_exp2_64).
// ---------------------------------------------------------------------------------------------
__constant__ double c_exp2_64[64] = {
    1.0, 1.0108892860517005, 1.0218971486541166, 1.0330248790212284,
    1.0442737824274138, 1.0556451783605572, 1.0671404006768237, 1.0787607977571199,
    1.0905077326652577, 1.102382583307841, 1.1143867425958924, 1.1265216186082418,
    1.1387886347566916, 1.1511892299529827, 1.1637248587775775, 1.1763969916502812,
    1.189207115002721, 1.202156731452703, 1.215247359980469, 1.22848053610687,
    1.241857812073484, 1.255380757024691, 1.2690509571917332, 1.2828700160787783,
    1.2968395546510096, 1.3109612115247644, 1.3252366431597413, 1.339667524053303,
    1.3542555469368927, 1.3690024229745905, 1.383909881963832, 1.3989796725383112,
    1.4142135623730951, 1.42961333839197, 1.4451808069770467, 1.460917794180647,
    1.4768261459394993, 1.4929077282912648, 1.5091644275934228, 1.5255981507445384,
    1.5422108254079407, 1.559004400237837, 1.5759808451078865, 1.593142151342267,
    1.6104903319492543, 1.6280274218573478, 1.645755478153965, 1.6636765803267364,
    1.681792830507429, 1.7001063537185235, 1.718619298122478, 1.7373338352737062,
    1.7562521603732995, 1.7753764925265212, 1.7947090750031072, 1.8142521755003989,
    1.8340080864093424, 1.8539791250833855, 1.8741676341103, 1.8945759815869656,
    1.9152065613971474, 1.9360617934922943, 1.9571441241754002, 1.978456026387951};

PIMD_DEV double exp_neg_tab64(double r2, const double *tab)
{
    const double MAGIC = 6755399441055744.0; // 1.5 * 2^52
    r2 = __hiloint2double(min(__double2hiint(r2), 0x40862000), __double2loint(r2)); // r2 <= 708 (r2 >= 0)
    const double t = fma(r2, -92.33248261689366, MAGIC); // -64 / ln 2
    const int j = __double2loint(t);
    const double kd = t - MAGIC;
    const double r = fma(kd, -0.010830424696249145, -r2); // ln2 / 64
    double p = 1.0 / 120.0;
    p = fma(p, r, 1.0 / 24.0);
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    const double v = tab[j & 63] * p;
    return __hiloint2double(__double2hiint(v) + (j >> 6) * 1048576, __double2loint(v));
}

// ---------------------------------------------------------------------------------------------
// The same with a 256-entry table (2 KB of shared memory): -r2 = j ln2/256 + r, |r| <= ln2/512,
// exp(-r2) = 2^(j>>8) * 2^((j&255)/256) * P4(r); degree-4 Taylor remainder r^5/120 <= 3.8e-17.
// 8 FP64 instructions.  Used by the pair kernel, whose rate is set by the FP64 instruction count.
// `tab` points to the 256 doubles 2^(i/256) in shared memory (copied from g_exp2_256).
// ---------------------------------------------------------------------------------------------
__device__ const double g_exp2_256[256] = {
    1.0, 1.0027112750502025, 1.0054299011128027, 1.0081558981184175,
    1.0108892860517005, 1.0136300849514894, 1.016378314910953, 1.019133996077738,
    1.0218971486541166, 1.0246677928971357, 1.0274459491187637, 1.030231637686041,
    1.0330248790212284, 1.0358256936019572, 1.0386341019613787, 1.041450124688316,
    1.0442737824274138, 1.0471050958792898, 1.0499440858006872, 1.0527907730046264,
    1.0556451783605572, 1.0585073227945128, 1.061377227289262, 1.0642549128844645,
    1.0671404006768237, 1.0700337118202419, 1.0729348675259756, 1.075843889062791,
    1.0787607977571199, 1.0816856149932152, 1.0846183622133092, 1.0875590609177697,
    1.0905077326652577, 1.0934643990728858, 1.0964290818163769, 1.099401802630222,
    1.102382583307841, 1.1053714457017412, 1.1083684117236787, 1.1113735033448175,
    1.1143867425958924, 1.1174081515673693, 1.1204377524096067, 1.12347556733302,
    1.1265216186082418, 1.129575928566288, 1.1326385195987192, 1.1357094141578055,
    1.1387886347566916, 1.1418762039695616, 1.1449721444318042, 1.148076478840179,
    1.1511892299529827, 1.154310420590216, 1.1574400736337511, 1.1605782120274988,
    1.1637248587775775, 1.1668800369524817, 1.1700437696832502, 1.1732160801636373,
    1.1763969916502812, 1.1795865274628758, 1.182784710984341, 1.1859915656609938,
    1.189207115002721, 1.1924313825831512, 1.1956643920398273, 1.1989061670743806,
    1.202156731452703, 1.2054161090051239, 1.2086843236265816, 1.2119613992768012,
    1.215247359980469, 1.2185422298274085, 1.2218460329727576, 1.2251587936371455,
    1.22848053610687, 1.2318112847340759, 1.2351510639369334, 1.2384998981998165,
    1.241857812073484, 1.245224830175258, 1.2486009771892048, 1.2519862778663162,
    1.255380757024691, 1.2587844395497165, 1.2621973503942507, 1.2656195145788063,
    1.2690509571917332, 1.2724917033894028, 1.275941778396392, 1.2794012075056693,
    1.2828700160787783, 1.2863482295460256, 1.2898358734066657, 1.2933329732290895,
    1.2968395546510096, 1.3003556433796506, 1.3038812651919358, 1.3074164459346773,
    1.3109612115247644, 1.3145155879493546, 1.318079601266064, 1.3216532776031575,
    1.3252366431597413, 1.3288297242059544, 1.3324325470831615, 1.3360451382041458,
    1.339667524053303, 1.3432997311868353, 1.3469417862329458, 1.3505937158920345,
    1.3542555469368927, 1.3579273062129011, 1.3616090206382248, 1.365300717204012,
    1.3690024229745905, 1.3727141650876684, 1.3764359707545302, 1.380167867260238,
    1.383909881963832, 1.387662042298529, 1.3914243757719262, 1.3951969099662003,
    1.3989796725383112, 1.4027726912202048, 1.4065759938190154, 1.4103896082172707,
    1.4142135623730951, 1.4180478843204152, 1.4218926021691656, 1.4257477441054942,
    1.42961333839197, 1.433489413367789, 1.4373759974489824, 1.4412731191286257,
    1.4451808069770467, 1.449099089642035, 1.4530279958490526, 1.4569675544014438,
    1.460917794180647, 1.4648787441464057, 1.4688504333369818, 1.4728328908693675,
    1.4768261459394993, 1.4808302278224719, 1.4848451658727524, 1.488870989524397,
    1.4929077282912648, 1.4969554117672355, 1.5010140696264256, 1.5050837316234065,
    1.5091644275934228, 1.5132561874526098, 1.5173590411982147, 1.5214730189088146,
    1.5255981507445384, 1.529734466947287, 1.533881997840956, 1.5380407738316568,
    1.5422108254079407, 1.5463921831410214, 1.550584877685, 1.5547889397770887,
    1.559004400237837, 1.5632312899713576, 1.567469639965553, 1.5717194812923414,
    1.5759808451078865, 1.5802537626528246, 1.5845382652524937, 1.588834384317164,
    1.593142151342267, 1.597461597908627, 1.6017927556826934, 1.606135656416771,
    1.6104903319492543, 1.6148568142048607, 1.6192351351948637, 1.6236253270173289,
    1.6280274218573478, 1.632441451987275, 1.6368674497669644, 1.6413054476440063,
    1.645755478153965, 1.6502175739206177, 1.6546917676561943, 1.6591780921616162,
    1.6636765803267364, 1.6681872651305825, 1.6727101796415966, 1.6772453570178785,
    1.681792830507429, 1.6863526334483934, 1.6909247992693053, 1.6955093614893326,
    1.7001063537185235, 1.7047158096580513, 1.709337763100463, 1.713972247929926,
    1.718619298122478, 1.723278947746274, 1.7279512309618377, 1.732636182022311,
    1.7373338352737062, 1.7420442251551564, 1.746767386199169, 1.7515033530318782,
    1.7562521603732995, 1.761013843037584, 1.7657884359332727, 1.7705759740635547,
    1.7753764925265212, 1.7801900265154245, 1.785016611318935, 1.789856282321401,
    1.7947090750031072, 1.7995750249405351, 1.804454167806624, 1.809346539371032,
    1.8142521755003989, 1.8191711121586085, 1.8241033854070534, 1.8290490314048973,
    1.8340080864093424, 1.8389805867758937, 1.843966568958626, 1.8489660695104508,
    1.8539791250833855, 1.8590057724288205, 1.864046048397789, 1.8690999899412386,
    1.8741676341103, 1.8792490180565602, 1.8843441790323345, 1.8894531543909392,
    1.8945759815869656, 1.8997126981765553, 1.9048633418176741, 1.9100279502703899,
    1.9152065613971474, 1.9203992131630474, 1.925605943636125, 1.930826790987627,
    1.9360617934922943, 1.9413109895286405, 1.9465744175792332, 1.9518521162309783,
    1.9571441241754002, 1.9624504802089273, 1.9677712232331759, 1.9731063922552343,
    1.978456026387951, 1.9838201648502194, 1.9891988469672663, 1.9945921121709402};

PIMD_DEV double exp_neg_tab256(double r2, const double *tab)
{
    const double MAGIC = 6755399441055744.0; // 1.5 * 2^52
    r2 = __hiloint2double(min(__double2hiint(r2), 0x40862000), __double2loint(r2)); // r2 <= 708 (r2 >= 0)
    const double t = fma(r2, -369.3299304675746, MAGIC); // -256 / ln 2
    const int j = __double2loint(t);
    const double kd = t - MAGIC;
    const double r = fma(kd, -0.0027076061740622863, -r2); // ln2 / 256
    double p = 1.0 / 24.0;
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    const double v = tab[j & 255] * p;
    return __hiloint2double(__double2hiint(v) + (j >> 8) * 1048576, __double2loint(v));
}

// exp(x) for any x through the same table: x is capped at 700 so that a wildly wrong exponent (a gauge that no
// longer fits) gives ~1e304 and trips the caller's range check instead of wrapping the exponent field
PIMD_DEV double exp_cap_tab64(double x, const double *tab)
{
    // x > 700 (or +NaN) -> 700, decided on the high word with integer compares (off the FP64 pipe)
    const bool big = __double2hiint(x) > 0x4085e000;
    return exp_neg_tab64(-__hiloint2double(big ? 0x4085e000 : __double2hiint(x), big ? 0 : __double2loint(x)), tab);
}

// exp(x) for any x through the 256-entry table (8 FP64 instructions), same cap as exp_cap_tab64
PIMD_DEV double exp_cap_tab256(double x, const double *tab)
{
    const bool big = __double2hiint(x) > 0x4085e000;
    return exp_neg_tab256(-__hiloint2double(big ? 0x4085e000 : __double2hiint(x), big ? 0 : __double2loint(x)), tab);
}

// ---------------------------------------------------------------------------------------------
// double-double helpers.  A dd value is (hi, lo) in a double2 (.x = hi, .y = lo).  The exchange
// tables a[u], q[l] reach 1e5..1e7 in magnitude while only their DIFFERENCES enter an exp, so
// they are carried as dd and differenced before rounding to double.
// ---------------------------------------------------------------------------------------------
PIMD_DEV double2 dd_add_d(double2 a, double b) // a + b, b a plain double
{
    double s = a.x + b;
    double bb = s - a.x;
    double e = (a.x - (s - bb)) + (b - bb); // TwoSum error
    e += a.y;
    double hi = s + e;
    double lo = e - (hi - s);
    return make_double2(hi, lo);
}
PIMD_DEV double2 dd_sub(double2 a, double2 b) // a - b as dd
{
    double s = a.x - b.x;
    double bb = s - a.x;
    double e = (a.x - (s - bb)) + (-b.x - bb);
    e += (a.y - b.y);
    double hi = s + e;
    double lo = e - (hi - s);
    return make_double2(hi, lo);
}
PIMD_DEV double dd_diff(double2 a, double2 b) // (a - b) rounded to double
{
    return (a.x - b.x) + (a.y - b.y);
}

// ---------------------------------------------------------------------------------------------
// signed log-sum-exp accumulator: sum_i sg_i exp(t_i) = s * exp(m), m = running max of t_i.
// ---------------------------------------------------------------------------------------------
struct Lse {
    double m, s;
};
PIMD_DEV Lse lse_empty() { return Lse{-INFINITY, 0.0}; }
PIMD_DEV void lse_shift(Lse &a, double delta) // re-reference: all t_i -> t_i + delta
{
    if (a.m != -INFINITY) a.m += delta;
}

// broadcast of a double from lane `src`: the two halves are shuffled separately and reassembled in
// place (a plain 64-bit __shfl_sync made ptxas swap the halves with three dependent XORs per use)
PIMD_DEV double shfl_bcast(double v, int src)
{
    const int lo = __shfl_sync(0xffffffffu, __double2loint(v), src);
    const int hi = __shfl_sync(0xffffffffu, __double2hiint(v), src);
    return __hiloint2double(hi, lo);
}

PIMD_DEV double shfl_xor_d(double v, int mask)
{
    const int lo = __shfl_xor_sync(0xffffffffu, __double2loint(v), mask);
    const int hi = __shfl_xor_sync(0xffffffffu, __double2hiint(v), mask);
    return __hiloint2double(hi, lo);
}

// warp reductions (all 32 lanes participate)
PIMD_DEV double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, shfl_xor_d(v, o));
    return v;
}
PIMD_DEV double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += shfl_xor_d(v, o);
    return v;
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11): counter (dof_lo, dof_hi, step_lo, step_hi), key
// (seed_lo, seed_hi); 53-bit uniforms from word pairs; Box-Muller.  z0 opens MD step `step`,
// z1 closes it.
// ---------------------------------------------------------------------------------------------
PIMD_DEV void philox_normal(uint64_t seed, uint64_t dof, uint64_t step, double &z0, double &z1)
{
    uint32_t c0 = (uint32_t)dof, c1 = (uint32_t)(dof >> 32), c2 = (uint32_t)step, c3 = (uint32_t)(step >> 32);
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        uint32_t n0 = h1 ^ c1 ^ k0, n2 = h0 ^ c3 ^ k1;
        c0 = n0; c1 = l1; c2 = n2; c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    uint64_t a = ((uint64_t)c0 << 32) | c1, b = ((uint64_t)c2 << 32) | c3;
    double u1 = ((double)(a >> 11) + 0.5) * 0x1.0p-53;
    double u2 = ((double)(b >> 11) + 0.5) * 0x1.0p-53;
    double r = sqrt(-2.0 * log(u1));
    double sn, cs;
    sincos(6.283185307179586476925286766559 * u2, &sn, &cs);
    z0 = r * cs;
    z1 = r * sn;
}

} // namespace pimd
