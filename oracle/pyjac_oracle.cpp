// =================================================================================================
// pyjac-b200 ORACLE  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, scalar CPU implementation of what the hot path computes: the constant-pressure /
// constant-volume source terms f = dphi/dt (Eqs. 1-8) and the analytical
// Jacobian J = df/dphi (Eq. 9) in the reformulated state
// phi = [T, V|P, n_1..n_{Ns-1}].  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call this file.  It shares no source, header, table or
// helper with paper_1809_01029_b200/ (the CUDA product).
//
// The paper defers every rate law and the Jacobian derivation to a supplement that is not available
// (PAPER.md L110, L171); the rate laws below are the standard CHEMKIN forms restated in
// DESIGN.md "Readings" and the Jacobian is the chain rule of SURVEY.md 8c-4, written
// out in that order with dense per-reaction partial vectors (no blocking, no sparsity exploitation).
//
// Everything is templated on the number type so that the SAME source-term code can be
//   - run in double                (the oracle value),
//   - run in long double           (4th-order central finite differences: pin P3),
//   - run in std::complex<double>  (complex-step derivative: pin P4; branches select on Re()).
// Pins: tests/test_oracle_*.py.  No function here is "parity unpinned".
//
// Build: g++ -O2 -fno-fast-math -ffp-contract=off -fopenmp -shared -fPIC  (oracle/build.py)
// =================================================================================================
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double R_GAS = 8314.46261815324;   // J/(kmol K)   reading S1
const double P_ATM = 101325.0;            // Pa
enum { T_ELEM = 0, T_THIRD, T_LIND, T_TROE, T_SRI, T_PLOG, T_CHEB };
enum { CONP = 0, CONV = 1 };

typedef std::complex<double> cplx;
using std::exp; using std::log; using std::log10;   // so long double / complex overloads are found
inline double re(double x) { return x; }
inline double re(long double x) { return (double)x; }
inline double re(const cplx& x) { return x.real(); }

template <class T> T ipow(const T& x, int n) {   // integer power by repeated multiplication (c-2)
    T r = T(1.0);
    for (int i = 0; i < n; ++i) r = r * x;
    return r;
}

struct Mech {
    int ns, nr;
    std::vector<double> W, tmid, lo, hi;
    std::vector<int> reac_ptr, reac_sp, reac_nu, prod_ptr, prod_sp, prod_nu;
    std::vector<int> rev, type;
    std::vector<double> A, beta, Ta;
    std::vector<int> eff_ptr, eff_sp;
    std::vector<double> eff_val;
    std::vector<int> collider;
    std::vector<double> lowA, lowb, lowTa, troe;
    std::vector<int> troe_t2;
    std::vector<int> chem;                   // chemically-activated falloff (reading R8): k = k_0 F / (1 + P_r)
    std::vector<double> revA, revb, revTa;   // explicit reverse Arrhenius parameters (reading R9); revA = 0: k_r = k_f / K_c
    std::vector<double> sri;
    std::vector<int> plog_ptr;
    std::vector<double> plogP, plogA, plogb, plogTa;
    std::vector<int> cheb_ptr, cheb_nT, cheb_nP;
    std::vector<double> chebTmin, chebTmax, chebPmin, chebPmax, cheb_coef;

    // nu'_ki, nu''_ki of species k in reaction i (0 if absent)
    int nu_r(int i, int k) const { int s = 0; for (int j = reac_ptr[i]; j < reac_ptr[i + 1]; ++j) if (reac_sp[j] == k) s += reac_nu[j]; return s; }
    int nu_p(int i, int k) const { int s = 0; for (int j = prod_ptr[i]; j < prod_ptr[i + 1]; ++j) if (prod_sp[j] == k) s += prod_nu[j]; return s; }
    bool has_third_body(int i) const { return type[i] >= T_THIRD && type[i] <= T_SRI; }
    // third-body efficiency alpha_ik (default 1; single collider "(+X)": delta_kX)
    double alpha(int i, int k) const {
        if (collider[i] >= 0) return k == collider[i] ? 1.0 : 0.0;
        for (int j = eff_ptr[i]; j < eff_ptr[i + 1]; ++j) if (eff_sp[j] == k) return eff_val[j];
        return 1.0;
    }
};

// every intermediate of the path, per state
template <class T> struct Inter {
    std::vector<T> C, cp, h, s, g;            // [ns]  cp [J/kmol/K], h [J/kmol], s/R, g/(RT)
    std::vector<T> dcp;                       // [ns]  d cp / dT
    std::vector<T> kf, kr, Kc, M, Pr, F, c, Rf, Rr, q;   // [nr]
    std::vector<T> k0_kinf;                               // [nr] falloff: k_0 / k_inf (= dP_r/d[M])
    std::vector<T> dlnkf_dT, dlnkf_dP, dlnKc_dT;         // [nr]
    std::vector<T> wdot;                      // [ns]; wdot[ns-1] from mass conservation (reading A1)
    T Ctot, D, N, S, Tt, P, V;
    void resize(int ns, int nr) {
        for (auto* v : {&C, &cp, &h, &s, &g, &dcp, &wdot}) v->assign(ns, T(0.0));
        for (auto* v : {&kf, &kr, &Kc, &M, &Pr, &F, &c, &Rf, &Rr, &q, &dlnkf_dT, &dlnkf_dP, &dlnKc_dT, &k0_kinf}) v->assign(nr, T(0.0));
    }
};

// ---- Troe / SRI blending functions (c-2) and their derivatives (c-4 item 5) ---------------------
template <class T> struct Blend { T F, dF_dPr, dF_dT; };

template <class T> Blend<T> blend(const Mech& m, int i, const T& Tt, const T& Pr_in) {
    Blend<T> b; b.F = T(1.0); b.dF_dPr = T(0.0); b.dF_dT = T(0.0);
    const double ln10 = std::log(10.0);
    T Pr = re(Pr_in) > 1e-300 ? Pr_in : T(1e-300);            // reading S5
    if (m.type[i] == T_TROE) {
        const double a = m.troe[4 * i], T3 = m.troe[4 * i + 1], T1 = m.troe[4 * i + 2], T2 = m.troe[4 * i + 3];
        T Fc = (1.0 - a) * exp(-Tt / T3) + a * exp(-Tt / T1);
        T dFc = -(1.0 - a) / T3 * exp(-Tt / T3) - a / T1 * exp(-Tt / T1);
        if (m.troe_t2[i]) { Fc = Fc + exp(-T2 / Tt); dFc = dFc + (T2 / (Tt * Tt)) * exp(-T2 / Tt); }
        T L = log10(Pr), Lc = log10(Fc);
        T n = 0.75 - 1.27 * Lc;
        T Aa = L - 0.4 - 0.67 * Lc;
        T B = n - 0.14 * Aa;
        T f = Aa / B;
        T log10F = Lc / (1.0 + f * f);
        b.F = exp(ln10 * log10F);
        T dlogF_df = -2.0 * Lc * f / ((1.0 + f * f) * (1.0 + f * f));
        T df_dL = n / (B * B);
        T df_dLc = (-0.67 * B + 1.1762 * Aa) / (B * B);
        b.dF_dPr = b.F * dlogF_df * df_dL / Pr;                // dF/dPr = F ln10 dlog10F/dL * 1/(Pr ln10)
        b.dF_dT = b.F * (1.0 / (1.0 + f * f) + dlogF_df * df_dLc) * dFc / Fc;
    } else if (m.type[i] == T_SRI) {
        const double a = m.sri[5 * i], bb = m.sri[5 * i + 1], cc = m.sri[5 * i + 2], d = m.sri[5 * i + 3], e = m.sri[5 * i + 4];
        T L = log10(Pr);
        T X = 1.0 / (1.0 + L * L);
        T base = a * exp(-bb / Tt) + exp(-Tt / cc);
        T dbase = (a * bb / (Tt * Tt)) * exp(-bb / Tt) - exp(-Tt / cc) / cc;
        b.F = d * exp(X * log(base)) * exp(e * log(Tt));
        b.dF_dPr = b.F * log(base) * (-2.0 * L * X * X) / (Pr * ln10);
        b.dF_dT = b.F * (X * dbase / base + e / Tt);
    }
    return b;
}

// ---- source terms, Eqs. 3-8, with every intermediate -------------------------------------------
template <class T>
// CL_rates (test hook for the "approximate" Jacobian pin): when non-null the rate expressions see
// this value as the last species' concentration (held fixed instead of C_tot - sum C_k) and the third-body
// concentration of a mixture is written [M] = C_tot + sum_k (alpha_k - 1) C_k; D and everything else are unchanged.
void eval_source(const Mech& m, int mode, const T* phi, const T& param, T* f, Inter<T>& w, const T* CL_rates = nullptr) {
    const int ns = m.ns, nr = m.nr;
    const double ln10 = std::log(10.0);
    const T Tt = phi[0];
    const T V = (mode == CONP) ? phi[1] : param;
    const T P = (mode == CONP) ? param : phi[1];
    w.Tt = Tt; w.P = P; w.V = V;
    // a1: concentrations (Eq. 6-7; last species from the ideal-gas law L122; order: reading S6)
    w.Ctot = P / (R_GAS * Tt);
    T sumC = T(0.0);
    for (int k = 0; k < ns - 1; ++k) { w.C[k] = phi[2 + k] / V; sumC = sumC + w.C[k]; }
    w.C[ns - 1] = w.Ctot - sumC;
    const T CL_true = w.C[ns - 1];
    if (CL_rates) w.C[ns - 1] = *CL_rates;
    // a2: NASA-7 thermo (c-2), low range iff T <= T_mid (reading S3)
    const T lnT = log(Tt);
    for (int k = 0; k < ns; ++k) {
        const double* a = (re(Tt) <= m.tmid[k]) ? &m.lo[7 * k] : &m.hi[7 * k];
        T T2 = Tt * Tt, T3 = T2 * Tt, T4 = T3 * Tt;
        T cpR = a[0] + a[1] * Tt + a[2] * T2 + a[3] * T3 + a[4] * T4;
        T hRT = a[0] + a[1] * Tt / 2.0 + a[2] * T2 / 3.0 + a[3] * T3 / 4.0 + a[4] * T4 / 5.0 + a[5] / Tt;
        T sR = a[0] * lnT + a[1] * Tt + a[2] * T2 / 2.0 + a[3] * T3 / 3.0 + a[4] * T4 / 4.0 + a[6];
        w.cp[k] = R_GAS * cpR;
        w.dcp[k] = R_GAS * (a[1] + 2.0 * a[2] * Tt + 3.0 * a[3] * T2 + 4.0 * a[4] * T3);
        w.h[k] = R_GAS * Tt * hRT;
        w.s[k] = sR;
        w.g[k] = hRT - sR;
    }
    // a3-a6: rate constants, pressure modification, rates of progress
    for (int i = 0; i < nr; ++i) {
        const int ty = m.type[i];
        T kf, lam_f, dlnk_dP = T(0.0);
        if (ty == T_PLOG) {
            // Entries with EQUAL pressures form one pressure LEVEL whose rate constant is the SUM of the entries'
            // Arrhenius rates (reading R10, the CHEMKIN convention for several P-Log lines per pressure); ln k is
            // interpolated linearly in ln P between neighbouring levels, constant outside the table (S4).
            const int p0 = m.plog_ptr[i], np_ = m.plog_ptr[i + 1] - p0;
            std::vector<int> first;                                   // first entry of every level, then np_
            for (int j = 0; j < np_; ++j) if (j == 0 || m.plogP[p0 + j] != m.plogP[p0 + j - 1]) first.push_back(j);
            const int nl = (int)first.size();
            first.push_back(np_);
            auto level = [&](int l, T& lnk, T& lam) {                  // ln k and d ln k / dT of level l
                auto lnk1 = [&](int j) { return std::log(m.plogA[p0 + j]) + m.plogb[p0 + j] * lnT - m.plogTa[p0 + j] / Tt; };
                auto lam1 = [&](int j) { return (m.plogb[p0 + j] + m.plogTa[p0 + j] / Tt) / Tt; };
                if (first[l + 1] - first[l] == 1) { lnk = lnk1(first[l]); lam = lam1(first[l]); return; }
                T ksum = T(0.0), dsum = T(0.0);
                for (int j = first[l]; j < first[l + 1]; ++j) { T kj = exp(lnk1(j)); ksum += kj; dsum += kj * lam1(j); }
                lnk = log(ksum); lam = dsum / ksum;
            };
            auto Pl = [&](int l) { return m.plogP[p0 + first[l]]; };
            const double Pre = re(P);
            T l0, lam0;
            if (Pre <= Pl(0)) { level(0, l0, lam0); kf = exp(l0); lam_f = lam0; }
            else if (Pre >= Pl(nl - 1)) { level(nl - 1, l0, lam0); kf = exp(l0); lam_f = lam0; }
            else {
                int j = 0;
                while (j + 2 < nl && Pl(j + 1) <= Pre) ++j;            // last level with P_j <= P (S4)
                const double dlnP = std::log(Pl(j + 1)) - std::log(Pl(j));
                T wgt = (log(P) - std::log(Pl(j))) / dlnP;
                T l1, lam1v;
                level(j, l0, lam0); level(j + 1, l1, lam1v);
                kf = exp(l0 + (l1 - l0) * wgt);
                lam_f = (1.0 - wgt) * lam0 + wgt * lam1v;
                dlnk_dP = (l1 - l0) / (dlnP * P);
            }
        } else if (ty == T_CHEB) {
            const int nT = m.cheb_nT[i], nP = m.cheb_nP[i];
            const double* eta = &m.cheb_coef[m.cheb_ptr[i]];
            const double iTmin = 1.0 / m.chebTmin[i], iTmax = 1.0 / m.chebTmax[i];
            const double lPmin = std::log10(m.chebPmin[i]), lPmax = std::log10(m.chebPmax[i]);
            T Tr = (2.0 / Tt - iTmin - iTmax) / (iTmax - iTmin);
            T Pr_ = (2.0 * log10(P) - lPmin - lPmax) / (lPmax - lPmin);
            std::vector<T> cT(nT), dT(nT), cP(nP), dP(nP);     // T_n and T_n' by the three-term recurrence
            for (int n = 0; n < nT; ++n) {
                if (n == 0) { cT[0] = T(1.0); dT[0] = T(0.0); }
                else if (n == 1) { cT[1] = Tr; dT[1] = T(1.0); }
                else { cT[n] = 2.0 * Tr * cT[n - 1] - cT[n - 2]; dT[n] = 2.0 * cT[n - 1] + 2.0 * Tr * dT[n - 1] - dT[n - 2]; }
            }
            for (int n = 0; n < nP; ++n) {
                if (n == 0) { cP[0] = T(1.0); dP[0] = T(0.0); }
                else if (n == 1) { cP[1] = Pr_; dP[1] = T(1.0); }
                else { cP[n] = 2.0 * Pr_ * cP[n - 1] - cP[n - 2]; dP[n] = 2.0 * cP[n - 1] + 2.0 * Pr_ * dP[n - 1] - dP[n - 2]; }
            }
            T lg = T(0.0), dlg_dTr = T(0.0), dlg_dPr = T(0.0);
            for (int a = 0; a < nT; ++a)
                for (int b = 0; b < nP; ++b) {
                    lg = lg + eta[a * nP + b] * cT[a] * cP[b];
                    dlg_dTr = dlg_dTr + eta[a * nP + b] * dT[a] * cP[b];
                    dlg_dPr = dlg_dPr + eta[a * nP + b] * cT[a] * dP[b];
                }
            kf = exp(ln10 * lg);
            lam_f = ln10 * dlg_dTr * (-2.0 / (Tt * Tt * (iTmax - iTmin)));
            dlnk_dP = dlg_dPr * 2.0 / (P * (lPmax - lPmin));    // ln10 * dlog10k/dPr~ * 2/(P ln10 (lPmax-lPmin))
        } else {
            kf = exp(std::log(m.A[i]) + m.beta[i] * lnT - m.Ta[i] / Tt);      // Arrhenius (c-2)
            lam_f = (m.beta[i] + m.Ta[i] / Tt) / Tt;
        }
        // Chemically-activated bimolecular reaction (reading R8): (A, beta, Ta) is still the
        // high-pressure limit k_inf and `low` the low-pressure limit k_0, P_r = k_0 [M] / k_inf as for falloff, but
        // the rate constant of the rates of progress is k_0 and the pressure modification is c = F / (1 + P_r).
        const bool chem = (ty == T_LIND || ty == T_TROE || ty == T_SRI) && m.chem[i];
        const T kinf = kf;
        if (chem) {
            kf = exp(std::log(m.lowA[i]) + m.lowb[i] * lnT - m.lowTa[i] / Tt);
            lam_f = (m.lowb[i] + m.lowTa[i] / Tt) / Tt;
        }
        w.kf[i] = kf; w.dlnkf_dT[i] = lam_f; w.dlnkf_dP[i] = dlnk_dP;
        // a4: equilibrium constant from Gibbs polynomials, reverse rate constant
        T kr = T(0.0), Kc = T(0.0), dlnKc = T(0.0);
        if (m.rev[i]) {
            T dg = T(0.0), dh = T(0.0); int snu = 0;
            for (int k = 0; k < ns; ++k) {
                int nu = m.nu_p(i, k) - m.nu_r(i, k);
                if (nu == 0) continue;
                dg = dg + double(nu) * w.g[k];
                dh = dh + double(nu) * w.h[k];
                snu += nu;
            }
            Kc = exp(-dg);
            T pf = P_ATM / (R_GAS * Tt);
            if (snu > 0) Kc = Kc * ipow(pf, snu);
            if (snu < 0) Kc = Kc / ipow(pf, -snu);
            kr = kf / Kc;
            dlnKc = dh / (R_GAS * Tt * Tt) - double(snu) / Tt;
            if (m.revA[i] > 0.0) {      // explicit reverse parameters (reading R9): K_c plays no role; the slot keeps k_f / k_r
                kr = exp(std::log(m.revA[i]) + m.revb[i] * lnT - m.revTa[i] / Tt);
                Kc = kf / kr;
                dlnKc = lam_f - (m.revb[i] + m.revTa[i] / Tt) / Tt;
            }
        }
        w.kr[i] = kr; w.Kc[i] = Kc; w.dlnKc_dT[i] = dlnKc;
        // a6: rates of progress by repeated multiplication
        T Rf = kf, Rr = kr;
        for (int j = m.reac_ptr[i]; j < m.reac_ptr[i + 1]; ++j) Rf = Rf * ipow(w.C[m.reac_sp[j]], m.reac_nu[j]);
        for (int j = m.prod_ptr[i]; j < m.prod_ptr[i + 1]; ++j) Rr = Rr * ipow(w.C[m.prod_sp[j]], m.prod_nu[j]);
        w.Rf[i] = Rf; w.Rr[i] = Rr;
        // a5: pressure modification c_i
        T c = T(1.0), M = T(0.0), Pr = T(0.0), F = T(1.0);
        if (m.has_third_body(i)) {
            if (CL_rates && m.collider[i] < 0) { M = w.Ctot; for (int k = 0; k < ns; ++k) M = M + (m.alpha(i, k) - 1.0) * w.C[k]; }
            else for (int k = 0; k < ns; ++k) M = M + m.alpha(i, k) * w.C[k];
            if (ty == T_THIRD) c = M;
            else {
                T k0 = exp(std::log(m.lowA[i]) + m.lowb[i] * lnT - m.lowTa[i] / Tt);
                w.k0_kinf[i] = k0 / kinf;
                Pr = k0 * M / kinf;
                F = blend(m, i, Tt, Pr).F;
                c = chem ? F / (1.0 + Pr) : F * Pr / (1.0 + Pr);
            }
        }
        w.M[i] = M; w.Pr[i] = Pr; w.F[i] = F; w.c[i] = c;
        w.q[i] = c * (Rf - Rr);                                   // Eq. 4
    }
    w.C[ns - 1] = CL_true;
    // a7: production rates (Eq. 4), last species by mass conservation (L122, reading A1)
    for (int k = 0; k < ns - 1; ++k) {
        T s = T(0.0);
        for (int i = 0; i < nr; ++i) {
            int nu = m.nu_p(i, k) - m.nu_r(i, k);
            if (nu != 0) s = s + double(nu) * w.q[i];
        }
        w.wdot[k] = s;
    }
    T ms = T(0.0);
    for (int k = 0; k < ns - 1; ++k) ms = ms + m.W[k] * w.wdot[k];
    w.wdot[ns - 1] = -ms / m.W[ns - 1];
    // Eq. 5: dT/dt
    T N = T(0.0), D = T(0.0), S = T(0.0);
    for (int k = 0; k < ns; ++k) {
        T Ek = (mode == CONP) ? w.h[k] : w.h[k] - R_GAS * Tt;
        T ck = (mode == CONP) ? w.cp[k] : w.cp[k] - R_GAS;
        N = N + Ek * w.wdot[k];
        D = D + w.C[k] * ck;
    }
    for (int k = 0; k < ns - 1; ++k) S = S + (1.0 - m.W[k] / m.W[ns - 1]) * w.wdot[k];
    w.N = N; w.D = D; w.S = S;
    f[0] = -N / D;
    // Eq. 8
    if (mode == CONP) f[1] = V * (Tt * R_GAS / P * S + f[0] / Tt);
    else f[1] = Tt * R_GAS * S + (P / Tt) * f[0];
    // Eq. 3
    for (int k = 0; k < ns - 1; ++k) f[2 + k] = V * w.wdot[k];
}

// ---- analytical Jacobian, dense, row-major nvar x nvar ------------------
// approx: the paper's "approximate" Jacobian (R6): in the species columns the
// derivatives of q_i through the last species' concentration are ignored, with [M] = C_tot + sum (alpha_k - 1) C_k.
void eval_jacobian(const Mech& m, int mode, bool approx, const double* phi, double param, double* J, Inter<double>& w) {
    const int ns = m.ns, nr = m.nr, nvar = ns + 1, L = ns - 1;
    std::vector<double> f(nvar);
    eval_source(m, mode, phi, param, f.data(), w);
    const double Tt = w.Tt, P = w.P, V = w.V, Ctot = w.Ctot;
    std::vector<double> G(ns), dq(nvar);
    std::vector<double> dW((size_t)(ns - 1) * nvar, 0.0);       // d wdot_k / d phi_c, k < Ns
    for (int i = 0; i < nr; ++i) {
        const int ty = m.type[i];
        const double R = w.Rf[i] - w.Rr[i];
        // item 3: mass-action partials
        std::vector<double> dRdC(ns, 0.0);
        for (int k = 0; k < ns; ++k) {
            int a = m.nu_r(i, k), b = m.nu_p(i, k);
            double t = 0.0;
            if (a > 0) {
                double pr = w.kf[i] * a;
                for (int j = m.reac_ptr[i]; j < m.reac_ptr[i + 1]; ++j) {
                    int l = m.reac_sp[j]; pr *= ipow(w.C[l], m.nu_r(i, l) - (l == k ? 1 : 0));
                }
                t += pr;
            }
            if (b > 0 && m.rev[i]) {
                double pr = w.kr[i] * b;
                for (int j = m.prod_ptr[i]; j < m.prod_ptr[i + 1]; ++j) {
                    int l = m.prod_sp[j]; pr *= ipow(w.C[l], m.nu_p(i, l) - (l == k ? 1 : 0));
                }
                t -= pr;
            }
            dRdC[k] = t;
        }
        const double lam_f = w.dlnkf_dT[i], lam_r = lam_f - w.dlnKc_dT[i];
        const double dRdT = lam_f * w.Rf[i] - lam_r * w.Rr[i];
        // item 4: partials of q_i = Q_i(T, P, C_1..C_Ns) by type
        double GT, GP = w.c[i] * w.dlnkf_dP[i] * R;
        double Xdef = 0.0;      // dQ_i/d[M] for a mixture third body: the part of G^k common to all default-efficiency species
        if (ty == T_THIRD) {
            if (m.collider[i] < 0) Xdef = R;
            for (int k = 0; k < ns; ++k) G[k] = m.alpha(i, k) * R + w.M[i] * dRdC[k];
            GT = w.M[i] * dRdT;
        } else if (ty == T_LIND || ty == T_TROE || ty == T_SRI) {
            const double Pr = w.Pr[i], F = w.F[i];
            Blend<double> b = blend(m, i, Tt, Pr);
            // c = F Pr / (1 + Pr) (falloff) or F / (1 + Pr) (chemically activated): dc/dPr at constant T, and the
            // factor of dF/dT
            const bool chem = m.chem[i] != 0;
            const double dc_dPr = chem ? -F / ((1.0 + Pr) * (1.0 + Pr)) + b.dF_dPr / (1.0 + Pr)
                                       : F / ((1.0 + Pr) * (1.0 + Pr)) + (Pr / (1.0 + Pr)) * b.dF_dPr;
            const double cF = chem ? 1.0 / (1.0 + Pr) : Pr / (1.0 + Pr);
            const double rat = w.k0_kinf[i];                              // dPr/d[M]
            const double dPr_dT = Pr * (m.lowb[i] - m.beta[i] + (m.lowTa[i] - m.Ta[i]) / Tt) / Tt;
            if (m.collider[i] < 0) Xdef = dc_dPr * rat * R;
            for (int k = 0; k < ns; ++k) G[k] = m.alpha(i, k) * dc_dPr * rat * R + w.c[i] * dRdC[k];
            GT = (dc_dPr * dPr_dT + cF * b.dF_dT) * R + w.c[i] * dRdT;
        } else {
            for (int k = 0; k < ns; ++k) G[k] = dRdC[k];
            GT = dRdT;
        }
        // items 1-2: chain rule from (T, P, C) to the state variables
        dq[0] = GT - (Ctot / Tt) * G[L];
        if (mode == CONP) {
            double s = 0.0;
            for (int k = 0; k < L; ++k) s += w.C[k] * (G[k] - G[L]);
            dq[1] = -s / V;
        } else {
            dq[1] = GP + G[L] / (R_GAS * Tt);
        }
        for (int j = 0; j < L; ++j) dq[2 + j] = approx ? (G[j] - Xdef) / V : (G[j] - G[L]) / V;
        for (int k = 0; k < L; ++k) {
            int nu = m.nu_p(i, k) - m.nu_r(i, k);
            if (nu == 0) continue;
            for (int c = 0; c < nvar; ++c) dW[(size_t)k * nvar + c] += double(nu) * dq[c];
        }
    }
    std::fill(J, J + (size_t)nvar * nvar, 0.0);
    // item 6: species rows, f_k = V wdot_k
    for (int k = 0; k < L; ++k)
        for (int c = 0; c < nvar; ++c) {
            double v = V * dW[(size_t)k * nvar + c];
            if (mode == CONP && c == 1) v += w.wdot[k];
            J[(size_t)(2 + k) * nvar + c] = v;
        }
    // item 7: T row and E row
    const double WL = m.W[L];
    auto En = [&](int k) { return mode == CONP ? w.h[k] : w.h[k] - R_GAS * Tt; };
    auto cn = [&](int k) { return mode == CONP ? w.cp[k] : w.cp[k] - R_GAS; };
    const double fT = f[0], fE = f[1], D = w.D, S = w.S;
    for (int c = 0; c < nvar; ++c) {
        double dN = 0.0, dS = 0.0;
        for (int k = 0; k < L; ++k) {
            dN += (En(k) - (m.W[k] / WL) * En(L)) * dW[(size_t)k * nvar + c];
            dS += (1.0 - m.W[k] / WL) * dW[(size_t)k * nvar + c];
        }
        double dD;
        if (c == 0) {
            for (int k = 0; k < L; ++k) dN += (cn(k) - (m.W[k] / WL) * cn(L)) * w.wdot[k];
            dD = 0.0;
            for (int k = 0; k < ns; ++k) dD += w.C[k] * w.dcp[k];
            dD -= cn(L) * Ctot / Tt;
        } else if (c == 1) {
            dD = (mode == CONP) ? -(D - Ctot * cn(L)) / V : cn(L) / (R_GAS * Tt);
        } else {
            dD = (cn(c - 2) - cn(L)) / V;
        }
        const double JT = -(dN + fT * dD) / D;
        J[c] = JT;
        double JE;
        if (mode == CONP) {
            JE = V * (Tt * R_GAS / P * dS + JT / Tt);
            if (c == 0) JE += V * (R_GAS * S / P - fT / (Tt * Tt));
            if (c == 1) JE += fE / V;
        } else {
            JE = Tt * R_GAS * dS + (P / Tt) * JT;
            if (c == 0) JE += R_GAS * S - P * fT / (Tt * Tt);
            if (c == 1) JE += fT / Tt;
        }
        J[(size_t)nvar + c] = JE;
    }
}

// ---- sparsity pattern, SURVEY.md 8c-5 ---------------------------------------
void pattern_dense_mask(const Mech& m, bool approx, std::vector<uint8_t>& mask) {
    const int ns = m.ns, nvar = ns + 1, L = ns - 1;
    mask.assign((size_t)nvar * nvar, 0);
    for (int c = 0; c < nvar; ++c) { mask[c] = 1; mask[(size_t)nvar + c] = 1; }           // rows T, E dense
    for (int r = 0; r < nvar; ++r) { mask[(size_t)r * nvar] = 1; mask[(size_t)r * nvar + 1] = 1; }   // columns T, E dense (S10)
    for (int i = 0; i < m.nr; ++i) {
        auto dep = [&](int k) { return m.nu_r(i, k) > 0 || (m.rev[i] && m.nu_p(i, k) > 0); };
        const bool depL = dep(L);
        for (int k = 0; k < L; ++k) {
            if (m.nu_p(i, k) - m.nu_r(i, k) == 0) continue;
            for (int j = 0; j < L; ++j) {
                bool in = approx ? (dep(j) || (m.has_third_body(i) && m.alpha(i, j) != (m.collider[i] >= 0 ? 0.0 : 1.0)))
                                 : (dep(j) || depL || (m.has_third_body(i) && m.alpha(i, j) != m.alpha(i, L)));
                if (in) mask[(size_t)(2 + k) * nvar + 2 + j] = 1;
            }
        }
    }
}

struct Handle {
    Mech m;
    bool approx = false;
    std::vector<uint8_t> mask;
    std::vector<int> csr_ptr, csr_idx, csc_ptr, csc_idx;
};

template <class V> void copy_in(std::vector<V>& dst, const V* src, size_t n) { dst.assign(src, src + n); }

}  // namespace

extern "C" {

struct orc_desc {
    int32_t n_species, n_reactions;
    const double *mol_weight, *nasa_tmid, *nasa_lo, *nasa_hi;
    const int32_t *reac_ptr, *reac_species, *reac_nu, *prod_ptr, *prod_species, *prod_nu;
    const uint8_t* reversible; const int32_t* type;
    const double *A, *beta, *Ta;
    const int32_t *eff_ptr, *eff_species; const double* eff_value;
    const int32_t* collider;
    const double *low_A, *low_beta, *low_Ta, *troe; const uint8_t* troe_has_T2; const double* sri;
    const int32_t* plog_ptr; const double *plog_P, *plog_A, *plog_beta, *plog_Ta;
    const int32_t *cheb_ptr, *cheb_nT, *cheb_nP;
    const double *cheb_Tmin, *cheb_Tmax, *cheb_Pmin, *cheb_Pmax, *cheb_coef;
    const uint8_t* chem_activated;            // [Nr] or NULL
    const double *rev_A, *rev_beta, *rev_Ta;  // [Nr] or NULL; rev_A > 0: explicit reverse rate constant
};

void* orc_create2(const orc_desc* d, int approx) {
    Handle* h = new Handle();
    h->approx = approx != 0;
    Mech& m = h->m;
    const int ns = d->n_species, nr = d->n_reactions;
    m.ns = ns; m.nr = nr;
    copy_in(m.W, d->mol_weight, ns); copy_in(m.tmid, d->nasa_tmid, ns);
    copy_in(m.lo, d->nasa_lo, 7 * ns); copy_in(m.hi, d->nasa_hi, 7 * ns);
    copy_in(m.reac_ptr, d->reac_ptr, nr + 1); copy_in(m.reac_sp, d->reac_species, d->reac_ptr[nr]); copy_in(m.reac_nu, d->reac_nu, d->reac_ptr[nr]);
    copy_in(m.prod_ptr, d->prod_ptr, nr + 1); copy_in(m.prod_sp, d->prod_species, d->prod_ptr[nr]); copy_in(m.prod_nu, d->prod_nu, d->prod_ptr[nr]);
    m.rev.resize(nr); for (int i = 0; i < nr; ++i) m.rev[i] = d->reversible[i];
    copy_in(m.type, d->type, nr);
    copy_in(m.A, d->A, nr); copy_in(m.beta, d->beta, nr); copy_in(m.Ta, d->Ta, nr);
    copy_in(m.eff_ptr, d->eff_ptr, nr + 1); copy_in(m.eff_sp, d->eff_species, d->eff_ptr[nr]); copy_in(m.eff_val, d->eff_value, d->eff_ptr[nr]);
    copy_in(m.collider, d->collider, nr);
    copy_in(m.lowA, d->low_A, nr); copy_in(m.lowb, d->low_beta, nr); copy_in(m.lowTa, d->low_Ta, nr);
    copy_in(m.troe, d->troe, 4 * nr); m.troe_t2.resize(nr); for (int i = 0; i < nr; ++i) m.troe_t2[i] = d->troe_has_T2[i];
    copy_in(m.sri, d->sri, 5 * nr);
    m.revA.assign(nr, 0.0); m.revb.assign(nr, 0.0); m.revTa.assign(nr, 0.0);
    if (d->rev_A) { copy_in(m.revA, d->rev_A, nr); copy_in(m.revb, d->rev_beta, nr); copy_in(m.revTa, d->rev_Ta, nr); }
    m.chem.assign(nr, 0); if (d->chem_activated) for (int i = 0; i < nr; ++i) m.chem[i] = d->chem_activated[i];
    copy_in(m.plog_ptr, d->plog_ptr, nr + 1);
    copy_in(m.plogP, d->plog_P, d->plog_ptr[nr]); copy_in(m.plogA, d->plog_A, d->plog_ptr[nr]);
    copy_in(m.plogb, d->plog_beta, d->plog_ptr[nr]); copy_in(m.plogTa, d->plog_Ta, d->plog_ptr[nr]);
    copy_in(m.cheb_ptr, d->cheb_ptr, nr + 1); copy_in(m.cheb_nT, d->cheb_nT, nr); copy_in(m.cheb_nP, d->cheb_nP, nr);
    copy_in(m.chebTmin, d->cheb_Tmin, nr); copy_in(m.chebTmax, d->cheb_Tmax, nr);
    copy_in(m.chebPmin, d->cheb_Pmin, nr); copy_in(m.chebPmax, d->cheb_Pmax, nr);
    copy_in(m.cheb_coef, d->cheb_coef, d->cheb_ptr[nr]);
    pattern_dense_mask(m, h->approx, h->mask);
    const int nvar = ns + 1;
    h->csr_ptr.assign(1, 0); h->csc_ptr.assign(1, 0);
    for (int r = 0; r < nvar; ++r) {
        for (int c = 0; c < nvar; ++c) if (h->mask[(size_t)r * nvar + c]) h->csr_idx.push_back(c);
        h->csr_ptr.push_back((int)h->csr_idx.size());
    }
    for (int c = 0; c < nvar; ++c) {
        for (int r = 0; r < nvar; ++r) if (h->mask[(size_t)r * nvar + c]) h->csc_idx.push_back(r);
        h->csc_ptr.push_back((int)h->csc_idx.size());
    }
    return h;
}

void* orc_create(const orc_desc* d) { return orc_create2(d, 0); }

void orc_destroy(void* hv) { delete (Handle*)hv; }

int64_t orc_nnz(void* hv) { return (int64_t)((Handle*)hv)->csr_idx.size(); }

// pattern: fmt 0 = CSR, 1 = CSC; ptr [nvar+1], idx [nnz]
void orc_pattern(void* hv, int fmt, int32_t* ptr, int32_t* idx) {
    Handle* h = (Handle*)hv;
    const std::vector<int>& p = fmt == 0 ? h->csr_ptr : h->csc_ptr;
    const std::vector<int>& x = fmt == 0 ? h->csr_idx : h->csc_idx;
    std::copy(p.begin(), p.end(), ptr); std::copy(x.begin(), x.end(), idx);
}

int orc_max_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// state-major inputs: phi [n][nvar], param [n]; out f [n][nvar]
void orc_source(void* hv, int mode, int64_t n, const double* phi, const double* param, double* f) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int nvar = m.ns + 1;
#pragma omp parallel
    {
        Inter<double> w; w.resize(m.ns, m.nr);
#pragma omp for schedule(static)
        for (int64_t s = 0; s < n; ++s) eval_source(m, mode, phi + s * nvar, param[s], f + s * nvar, w);
    }
}

// ---- conversions between the common mass / mole fractions and the paper's state vector ("conversion
// to/from the more-common mass/mole fractions and moles is straightforward"; Eq. 1).  Plain definitions:
//   mole fractions from mass fractions:  X_k = (Y_k / W_k) / sum_j (Y_j / W_j)
//   moles:                               n_k = X_k n_tot,  n_tot = P V / (R T)   (ideal-gas law), k = 1 .. Ns-1
//   back:                                X_k = n_k / n_tot (k < Ns), X_Ns = 1 - sum_{k<Ns} X_k  (the last species'
//                                        moles follow from the ideal-gas law);  Y_k = X_k W_k / sum_j X_j W_j
// kind 0: mole fractions, 1: mass fractions.  State-major arrays: frac [n][ns], phi [n][nvar], T, P, V, param [n].
void orc_state_from_fractions(void* hv, int mode, int kind, int64_t n, const double* Tt, const double* P, const double* V,
                              const double* frac, double* phi, double* param) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int ns = m.ns, nvar = ns + 1;
    for (int64_t s = 0; s < n; ++s) {
        std::vector<double> X(frac + s * ns, frac + (s + 1) * ns);
        if (kind == 1) {
            double sum = 0.0;
            for (int k = 0; k < ns; ++k) sum += frac[s * ns + k] / m.W[k];
            for (int k = 0; k < ns; ++k) X[k] = (frac[s * ns + k] / m.W[k]) / sum;
        }
        const double ntot = P[s] * V[s] / (R_GAS * Tt[s]);
        phi[s * nvar] = Tt[s];
        phi[s * nvar + 1] = mode == 0 ? V[s] : P[s];
        param[s] = mode == 0 ? P[s] : V[s];
        for (int k = 0; k < ns - 1; ++k) phi[s * nvar + 2 + k] = X[k] * ntot;
    }
}

void orc_fractions_from_state(void* hv, int mode, int kind, int64_t n, const double* phi, const double* param, double* frac) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int ns = m.ns, nvar = ns + 1;
    for (int64_t s = 0; s < n; ++s) {
        const double Tt = phi[s * nvar];
        const double V = mode == 0 ? phi[s * nvar + 1] : param[s], P = mode == 0 ? param[s] : phi[s * nvar + 1];
        const double ntot = P * V / (R_GAS * Tt);
        std::vector<double> X(ns);
        double sum = 0.0;
        for (int k = 0; k < ns - 1; ++k) { X[k] = phi[s * nvar + 2 + k] / ntot; sum += X[k]; }
        X[ns - 1] = 1.0 - sum;
        if (kind == 0) { for (int k = 0; k < ns; ++k) frac[s * ns + k] = X[k]; continue; }
        double wbar = 0.0;
        for (int k = 0; k < ns; ++k) wbar += X[k] * m.W[k];
        for (int k = 0; k < ns; ++k) frac[s * ns + k] = X[k] * m.W[k] / wbar;
    }
}

// J [n][nvar][nvar] row-major, entry (i,j) = d f_i / d phi_j  (Eq. 9)
void orc_jacobian_dense(void* hv, int mode, int64_t n, const double* phi, const double* param, double* J) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int nvar = m.ns + 1;
#pragma omp parallel
    {
        Inter<double> w; w.resize(m.ns, m.nr);
#pragma omp for schedule(static)
        for (int64_t s = 0; s < n; ++s) eval_jacobian(m, mode, h->approx, phi + s * nvar, param[s], J + (size_t)s * nvar * nvar, w);
    }
}

// vals [n][nnz] in CSR (fmt 0) or CSC (fmt 1) value order
void orc_jacobian_sparse(void* hv, int mode, int fmt, int64_t n, const double* phi, const double* param, double* vals) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int nvar = m.ns + 1;
    const size_t nnz = h->csr_idx.size();
#pragma omp parallel
    {
        Inter<double> w; w.resize(m.ns, m.nr);
        std::vector<double> J((size_t)nvar * nvar);
#pragma omp for schedule(static)
        for (int64_t s = 0; s < n; ++s) {
            eval_jacobian(m, mode, h->approx, phi + s * nvar, param[s], J.data(), w);
            double* o = vals + (size_t)s * nnz;
            size_t e = 0;
            if (fmt == 0) { for (int r = 0; r < nvar; ++r) for (int p = h->csr_ptr[r]; p < h->csr_ptr[r + 1]; ++p) o[e++] = J[(size_t)r * nvar + h->csr_idx[p]]; }
            else { for (int c = 0; c < nvar; ++c) for (int p = h->csc_ptr[c]; p < h->csc_ptr[c + 1]; ++p) o[e++] = J[(size_t)h->csc_idx[p] * nvar + c]; }
        }
    }
}

// every intermediate of one state; arrays sized [ns] or [nr]; scal = {Ctot, D, N, S}
void orc_intermediates(void* hv, int mode, const double* phi, double param, double* C, double* cp, double* hk, double* sk,
                       double* g, double* kf, double* kr, double* Kc, double* M, double* Pr, double* F, double* c,
                       double* Rf, double* Rr, double* q, double* wdot, double* scal) {
    Handle* h = (Handle*)hv; const Mech& m = h->m;
    Inter<double> w; w.resize(m.ns, m.nr);
    std::vector<double> f(m.ns + 1);
    eval_source(m, mode, phi, param, f.data(), w);
    auto cp_ = [](const std::vector<double>& v, double* o) { std::copy(v.begin(), v.end(), o); };
    cp_(w.C, C); cp_(w.cp, cp); cp_(w.h, hk); cp_(w.s, sk); cp_(w.g, g); cp_(w.kf, kf); cp_(w.kr, kr); cp_(w.Kc, Kc);
    cp_(w.M, M); cp_(w.Pr, Pr); cp_(w.F, F); cp_(w.c, c); cp_(w.Rf, Rf); cp_(w.Rr, Rr); cp_(w.q, q); cp_(w.wdot, wdot);
    scal[0] = w.Ctot; scal[1] = w.D; scal[2] = w.N; scal[3] = w.S;
}

// First-order forward finite-difference Jacobian, the paper's comparison baseline (Fig. 12), written
// out column by column in double.  The paper gives no step rule; R7:
//     xp_c = phi_c + fma(rel, |phi_c|, abs),  h_c = xp_c - phi_c,  J(i,c) = (f_i(phi; phi_c := xp_c) - f_i(phi)) / h_c.
// J [n][nvar][nvar] row-major.  Pinned against the analytical Jacobian (first-order convergence, test P13).
void orc_fd1_jacobian(void* hv, int mode, int64_t n, const double* phi, const double* param, double rel, double abs_, double* J) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int nvar = m.ns + 1;
#pragma omp parallel
    {
        Inter<double> w; w.resize(m.ns, m.nr);
        std::vector<double> x(nvar), f0(nvar), f1(nvar);
#pragma omp for schedule(static)
        for (int64_t s = 0; s < n; ++s) {
            const double* ph = phi + s * nvar;
            double* Js = J + (size_t)s * nvar * nvar;
            eval_source<double>(m, mode, ph, param[s], f0.data(), w);
            for (int c = 0; c < nvar; ++c) {
                for (int k = 0; k < nvar; ++k) x[k] = ph[k];
                const double xp = ph[c] + std::fma(rel, std::fabs(ph[c]), abs_);
                const double hc = xp - ph[c];
                x[c] = xp;
                eval_source<double>(m, mode, x.data(), param[s], f1.data(), w);
                for (int r = 0; r < nvar; ++r) Js[(size_t)r * nvar + c] = (f1[r] - f0[r]) / hc;
            }
        }
    }
}

// pin P3: 4th-order central finite differences of the oracle's own f, evaluated in long double.
// step h_c = rel * max(|phi_c|, floor_c); J row-major nvar x nvar (double)
void orc_fd_jacobian(void* hv, int mode, const double* phi, double param, double rel, const double* floor_, double* J) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int nvar = m.ns + 1;
    Inter<long double> w; w.resize(m.ns, m.nr);
    std::vector<long double> x(nvar), f1(nvar), f2(nvar), f3(nvar), f4(nvar);
    for (int c = 0; c < nvar; ++c) {
        long double hc = (long double)rel * std::max(std::fabs(phi[c]), floor_[c]);
        auto ev = [&](long double d, std::vector<long double>& f) {
            for (int k = 0; k < nvar; ++k) x[k] = phi[k];
            x[c] += d;
            eval_source<long double>(m, mode, x.data(), (long double)param, f.data(), w);
        };
        ev(-2 * hc, f1); ev(-hc, f2); ev(hc, f3); ev(2 * hc, f4);
        for (int r = 0; r < nvar; ++r) J[(size_t)r * nvar + c] = (double)((f1[r] - 8 * f2[r] + 8 * f3[r] - f4[r]) / (12 * hc));
    }
}

// pin P4: complex-step derivative, h_c = rel * max(|phi_c|, floor_c)
void orc_cs_jacobian(void* hv, int mode, const double* phi, double param, double rel, const double* floor_, double* J) {
    Handle* h = (Handle*)hv; const Mech& m = h->m; const int nvar = m.ns + 1;
    Inter<cplx> w; w.resize(m.ns, m.nr);
    std::vector<cplx> x(nvar), f(nvar);
    for (int c = 0; c < nvar; ++c) {
        double hc = rel * std::max(std::fabs(phi[c]), floor_[c]);
        for (int k = 0; k < nvar; ++k) x[k] = cplx(phi[k], 0.0);
        x[c] = cplx(phi[c], hc);
        if (h->approx && c >= 2) {          // approximate Jacobian: C_Ns held fixed inside the rates for the species columns
            double sum = 0.0;
            const double Vr = mode == CONP ? phi[1] : param, Pr = mode == CONP ? param : phi[1];
            for (int k = 0; k < m.ns - 1; ++k) sum += phi[2 + k] / Vr;
            const cplx CL(Pr / (R_GAS * phi[0]) - sum, 0.0);
            eval_source<cplx>(m, mode, x.data(), cplx(param, 0.0), f.data(), w, &CL);
        } else
        eval_source<cplx>(m, mode, x.data(), cplx(param, 0.0), f.data(), w);
        for (int r = 0; r < nvar; ++r) J[(size_t)r * nvar + c] = f[r].imag() / hc;
    }
}

}  // extern "C"
