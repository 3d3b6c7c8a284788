"""Oracle: aligned-spin PhenomD (2,2) mode and PhenomHM higher modes.

Follows SURVEY.md 8(c) O0-O3 (the paper only cites the model, PAPER.md:110-116,
eq. 5; t_lm(f) is eq. 6).  All frequencies inside this module are
dimensionless Mf unless a name ends in _hz.  Phase convention (O0):
h_lm(f) = A_lm(f) exp(i phi_lm(f)) with phi_lm = -Psi_lm, Psi the
TaylorF2-signed phase.  TEST INFRASTRUCTURE - see oracle/__init__.py.
"""
import math

import numpy as np

from .constants import EULER_GAMMA, GPC_S, MODES, MTSUN_S

PI = math.pi
F_AMP_INS = 0.014      # end of the inspiral amplitude region (Mf)
F_PHI_INS = 0.018      # end of the inspiral phase region (Mf)
COEF_NAMES = ("rho1", "rho2", "rho3", "v2", "gamma1", "gamma2", "gamma3",
              "sigma1", "sigma2", "sigma3", "sigma4", "beta1", "beta2", "beta3",
              "alpha1", "alpha2", "alpha3", "alpha4", "alpha5")


def fit_value(table, name, eta, chi_hat):
    """Bilinear-cubic fit form of O1: 11 numbers per coefficient."""
    x = chi_hat - 1.0
    g = lambda k: table[f"pd.{name}.{k}"]
    return (g("l00") + g("l10") * eta
            + x * (g("l01") + g("l11") * eta + g("l21") * eta * eta)
            + x * x * (g("l02") + g("l12") * eta + g("l22") * eta * eta)
            + x * x * x * (g("l03") + g("l13") * eta + g("l23") * eta * eta))


def final_spin(table, eta, S):
    g = lambda k: table[f"fs.spin.{k}"]
    S2, S3, S4 = S * S, S ** 3, S ** 4
    af = (2.0 * math.sqrt(3.0) * eta + g("e2") * eta ** 2 + g("e3") * eta ** 3 + g("e4") * eta ** 4
          + eta * (g("s1e1") * S + g("s2e1") * S2 + g("s3e1") * S3 + g("s4e1") * S4)
          + eta ** 2 * (g("s1e2") * S + g("s2e2") * S2 + g("s3e2") * S3 + g("s4e2") * S4)
          + S)
    return min(af, 0.999)          # DESIGN.md reading R-af: keep (1-a_f)^p real


def radiated_energy(table, eta, S_hat):
    g = lambda k: table[f"fs.erad.{k}"]
    num = eta * (g("e1") + g("e2") * eta + g("e3") * eta ** 2 + g("e4") * eta ** 3)
    return num * (1.0 + (g("n0") + g("n1") * eta + g("n2") * eta ** 2) * S_hat) / \
        (1.0 + (g("d0") + g("d1") * eta + g("d2") * eta ** 2) * S_hat)


class Intrinsic:
    """Step O1: everything that depends on {M_T, q, a1, a2, D_L} only."""

    def __init__(self, table, M_T, q, a1, a2, D_L):
        self.table = table
        qq = max(q, 1.0 / q)                       # G15: m1 >= m2, a1 belongs to m1
        m1 = qq / (1.0 + qq)
        m2 = 1.0 / (1.0 + qq)
        self.m1, self.m2 = m1, m2
        self.eta = eta = m1 * m2
        self.delta = delta = m1 - m2
        self.chi_s = chi_s = 0.5 * (a1 + a2)
        self.chi_a = chi_a = 0.5 * (a1 - a2)
        chi_eff = m1 * a1 + m2 * a2
        chi_pn = chi_eff - (38.0 * eta / 113.0) * (a1 + a2)
        self.chi_hat = chi_pn / (1.0 - 76.0 * eta / 113.0)
        self.M_s = M_T * MTSUN_S                   # geometric total mass in seconds
        self.amp0 = self.M_s ** 2 / (D_L * GPC_S)  # strain * seconds
        # final state and quasi-normal modes
        S = m1 * m1 * a1 + m2 * m2 * a2
        self.a_f = final_spin(table, eta, S)
        self.E_rad = radiated_energy(table, eta, S / (1.0 - 2.0 * eta))
        self.f_rd = {}
        self.f_damp = {}
        for (l, m) in MODES:
            g = lambda k: table[f"qnm.{l}{m}.{k}"]
            omega = g("f1") + g("f2") * (1.0 - self.a_f) ** g("f3")
            Q = g("q1") + g("q2") * (1.0 - self.a_f) ** g("q3")
            frd = omega / (2.0 * PI * (1.0 - self.E_rad))
            self.f_rd[(l, m)] = frd
            self.f_damp[(l, m)] = frd / (2.0 * Q)
        self.fRD = self.f_rd[(2, 2)]
        self.fDM = self.f_damp[(2, 2)]
        for name in COEF_NAMES:
            setattr(self, name, fit_value(table, name, eta, self.chi_hat))
        self._pn_phase()
        self._pn_amp()
        self._amp_setup()
        self._phase_setup()

    # ------------------------------------------------------------------ PN
    def _pn_phase(self):
        eta, d, xs, xa = self.eta, self.delta, self.chi_s, self.chi_a
        e2, e3 = eta * eta, eta ** 3
        self.ph = ph = [0.0] * 8
        ph[0] = 1.0
        ph[1] = 0.0
        ph[2] = 3715.0 / 756.0 + 55.0 * eta / 9.0
        ph[3] = -16.0 * PI + 113.0 * d * xa / 3.0 + (113.0 / 3.0 - 76.0 * eta / 3.0) * xs
        ph[4] = (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * e2 / 72.0
                 + (-405.0 / 8.0 + 200.0 * eta) * xa * xa - 405.0 / 4.0 * d * xa * xs
                 + (-405.0 / 8.0 + 5.0 * eta / 2.0) * xs * xs)
        # ph[5] multiplies [1 + ln(pi f)]
        ph[5] = (38645.0 * PI / 756.0 - 65.0 * PI * eta / 9.0
                 + d * (-732985.0 / 2268.0 - 140.0 * eta / 9.0) * xa
                 + (-732985.0 / 2268.0 + 24260.0 * eta / 81.0 + 340.0 * e2 / 9.0) * xs)
        # ph[6] is the constant part; the log part is -(6848/63) ln(64 pi f)
        ph[6] = (11583231236531.0 / 4694215680.0 - 6848.0 * EULER_GAMMA / 21.0 - 640.0 * PI * PI / 3.0
                 + (-15737765635.0 / 3048192.0 + 2255.0 * PI * PI / 12.0) * eta
                 + 76055.0 * e2 / 1728.0 - 127825.0 * e3 / 1296.0
                 + 2270.0 * PI / 3.0 * d * xa + (2270.0 * PI / 3.0 - 520.0 * PI * eta) * xs)
        ph[7] = (77096675.0 * PI / 254016.0 + 378515.0 * PI * eta / 1512.0 - 74045.0 * PI * e2 / 756.0
                 + d * (-25150083775.0 / 3048192.0 + 26804935.0 * eta / 6048.0 - 1985.0 * e2 / 48.0) * xa
                 + (-25150083775.0 / 3048192.0 + 10566655595.0 * eta / 762048.0
                    - 1042165.0 * e2 / 3024.0 + 5345.0 * e3 / 36.0) * xs)
        self.ph6_log = -6848.0 / 63.0

    def _pn_amp(self):
        eta, d, xs, xa = self.eta, self.delta, self.chi_s, self.chi_a
        e2, e3 = eta * eta, eta ** 3
        self.am = am = [0.0] * 7
        am[0] = 1.0
        am[1] = 0.0
        am[2] = -323.0 / 224.0 + 451.0 * eta / 168.0
        am[3] = 27.0 * d * xa / 8.0 + (27.0 / 8.0 - 11.0 * eta / 6.0) * xs
        am[4] = (-27312085.0 / 8128512.0 - 1975055.0 * eta / 338688.0 + 105271.0 * e2 / 24192.0
                 + (-81.0 / 32.0 + 8.0 * eta) * xa * xa - 81.0 / 16.0 * d * xa * xs
                 + (-81.0 / 32.0 + 17.0 * eta / 8.0) * xs * xs)
        am[5] = (-85.0 * PI / 64.0 + 85.0 * PI * eta / 16.0
                 + d * (285197.0 / 16128.0 - 1579.0 * eta / 4032.0) * xa
                 + (285197.0 / 16128.0 - 15317.0 * eta / 672.0 - 2227.0 * e2 / 1008.0) * xs)
        am[6] = (-177520268561.0 / 8583708672.0
                 + (545384828789.0 / 5007163392.0 - 205.0 * PI * PI / 48.0) * eta
                 - 3248849057.0 * e2 / 178827264.0 + 34473079.0 * e3 / 6386688.0
                 + (1614569.0 / 64512.0 - 1873643.0 * eta / 16128.0 + 2167.0 * e2 / 42.0) * xa * xa
                 + (31.0 * PI / 12.0 - 7.0 * PI * eta / 3.0) * xs
                 + (1614569.0 / 64512.0 - 61391.0 * eta / 1344.0 + 57451.0 * e2 / 4032.0) * xs * xs
                 + d * xa * (31.0 * PI / 12.0 + (1614569.0 / 32256.0 - 165961.0 * eta / 2688.0) * xs))

    # ----------------------------------------------------------- amplitude
    def amp_ins(self, f):
        """A-hat (amplitude / A0) in the inspiral region and its f-derivative."""
        f = np.asarray(f, dtype=np.float64)
        val = np.zeros_like(f)
        der = np.zeros_like(f)
        for i in range(7):
            c = self.am[i] * PI ** (i / 3.0)
            val = val + c * f ** (i / 3.0)
            if i > 0:
                der = der + c * (i / 3.0) * f ** (i / 3.0 - 1.0)
        val = val + self.rho1 * f ** (7.0 / 3.0) + self.rho2 * f ** (8.0 / 3.0) + self.rho3 * f ** 3
        der = der + (7.0 / 3.0) * self.rho1 * f ** (4.0 / 3.0) + (8.0 / 3.0) * self.rho2 * f ** (5.0 / 3.0) \
            + 3.0 * self.rho3 * f ** 2
        return val, der

    def amp_mr(self, f):
        """Merger-ringdown A-hat: Lorentzian times exponential (O2)."""
        f = np.asarray(f, dtype=np.float64)
        w = self.gamma3 * self.fDM
        x = f - self.fRD
        lor = 1.0 / (x * x + w * w)
        val = self.gamma1 * w * lor * np.exp(-self.gamma2 * x / w)
        der = val * (-2.0 * x * lor - self.gamma2 / w)
        return val, der

    def _amp_setup(self):
        g2, g3 = self.gamma2, self.gamma3
        if g2 >= 1.0:
            self.f_peak = abs(self.fRD - self.fDM * g3 / g2)
        else:
            self.f_peak = abs(self.fRD + self.fDM * g3 * (math.sqrt(1.0 - g2 * g2) - 1.0) / g2)
        f1, f3 = F_AMP_INS, self.f_peak
        f2 = 0.5 * (f1 + f3)
        v1, d1 = self.amp_ins(f1)
        v3, d3 = self.amp_mr(f3)
        # five collocation conditions for delta_0..delta_4 (values at f1,f2,f3; slopes at f1,f3)
        A = np.array([[1.0, f1, f1 ** 2, f1 ** 3, f1 ** 4],
                      [1.0, f2, f2 ** 2, f2 ** 3, f2 ** 4],
                      [1.0, f3, f3 ** 2, f3 ** 3, f3 ** 4],
                      [0.0, 1.0, 2 * f1, 3 * f1 ** 2, 4 * f1 ** 3],
                      [0.0, 1.0, 2 * f3, 3 * f3 ** 2, 4 * f3 ** 3]])
        b = np.array([float(v1), self.v2, float(v3), float(d1), float(d3)])
        self.delta_int = np.linalg.solve(A, b)
        # f_ref = argmax f^2 A_22(f): root of d/df ln(f^(5/6) A-hat_MR) above f_peak (G4)
        w = g3 * self.fDM

        def g(f):
            x = f - self.fRD
            return (5.0 / 6.0) / f - 2.0 * x / (x * x + w * w) - g2 / w

        lo, hi = self.f_peak, self.fRD + 4.0 * w
        while g(hi) > 0.0:
            hi += w
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if mid == lo or mid == hi:
                break
            if g(mid) > 0.0:
                lo = mid
            else:
                hi = mid
        self.f_ref = 0.5 * (lo + hi)

    def amp_hat(self, f):
        """A-hat(f) over all three regions (C1 by construction)."""
        f = np.asarray(f, dtype=np.float64)
        d = self.delta_int
        ins = self.amp_ins(f)[0]
        mid = d[0] + f * (d[1] + f * (d[2] + f * (d[3] + f * d[4])))
        mr = self.amp_mr(f)[0]
        return np.where(f < F_AMP_INS, ins, np.where(f < self.f_peak, mid, mr))

    def amp22(self, f):
        """|h_22(f)| in strain*seconds: amp0 * A0(f) * A-hat(f), A0 = sqrt(2 eta/3) pi^(-1/6) f^(-7/6)."""
        f = np.asarray(f, dtype=np.float64)
        A0 = math.sqrt(2.0 * self.eta / 3.0) * PI ** (-1.0 / 6.0) * f ** (-7.0 / 6.0)
        return self.amp0 * A0 * self.amp_hat(f)

    # --------------------------------------------------------------- phase
    def _psi_ins_raw(self, f):
        f = np.asarray(f, dtype=np.float64)
        eta = self.eta
        pf = PI * f
        lnpf = np.log(pf)
        ph = self.ph
        s = np.zeros_like(f)
        ds = np.zeros_like(f)
        for i in range(8):
            p = (i - 5.0) / 3.0
            if i == 5:
                c = ph[5] * (1.0 + lnpf)
                dc = ph[5] / f
            elif i == 6:
                c = ph[6] + self.ph6_log * np.log(64.0 * pf)
                dc = self.ph6_log / f
            else:
                c = ph[i]
                dc = 0.0
            term = pf ** p
            s = s + c * term
            ds = ds + dc * term + c * p * term / f
        pre = 3.0 / (128.0 * eta)
        psi = -PI / 4.0 + pre * s
        dpsi = pre * ds
        psi = psi + (self.sigma1 * f + 0.75 * self.sigma2 * f ** (4.0 / 3.0)
                     + 0.6 * self.sigma3 * f ** (5.0 / 3.0) + 0.5 * self.sigma4 * f * f) / eta
        dpsi = dpsi + (self.sigma1 + self.sigma2 * f ** (1.0 / 3.0)
                       + self.sigma3 * f ** (2.0 / 3.0) + self.sigma4 * f) / eta
        return psi, dpsi

    def _psi_int_raw(self, f):
        f = np.asarray(f, dtype=np.float64)
        psi = (self.beta1 * f + self.beta2 * np.log(f) - self.beta3 / 3.0 * f ** -3.0) / self.eta
        dpsi = (self.beta1 + self.beta2 / f + self.beta3 * f ** -4.0) / self.eta
        return psi, dpsi

    def _psi_mr_raw(self, f):
        f = np.asarray(f, dtype=np.float64)
        x = f - self.alpha5 * self.fRD
        psi = (self.alpha1 * f - self.alpha2 / f + 4.0 / 3.0 * self.alpha3 * f ** 0.75
               + self.alpha4 * np.arctan(x / self.fDM)) / self.eta
        dpsi = (self.alpha1 + self.alpha2 / (f * f) + self.alpha3 * f ** -0.25
                + self.alpha4 * self.fDM / (self.fDM ** 2 + x * x)) / self.eta
        return psi, dpsi

    def _phase_setup(self):
        self.f_mr = 0.5 * self.fRD
        # C1 connection constants (the fitted beta1/alpha1 are absorbed here, O2)
        p_i, dp_i = self._psi_ins_raw(F_PHI_INS)
        p_m, dp_m = self._psi_int_raw(F_PHI_INS)
        self.C2_int = float(dp_i - dp_m)
        self.C1_int = float(p_i - p_m - self.C2_int * F_PHI_INS)
        p_m2, dp_m2 = self._psi_int_raw(self.f_mr)
        p_m2 = p_m2 + self.C1_int + self.C2_int * self.f_mr
        dp_m2 = dp_m2 + self.C2_int
        p_r, dp_r = self._psi_mr_raw(self.f_mr)
        self.C2_mr = float(dp_m2 - dp_r)
        self.C1_mr = float(p_m2 - p_r - self.C2_mr * self.f_mr)
        # alignment (G4): Psi(f_ref) = 0 and Psi'(f_ref) = 0
        self.t_shift = 0.0
        self.p_shift = 0.0
        p0, dp0 = self.psi22(np.float64(self.f_ref))
        self.t_shift = float(dp0)
        self.p_shift = float(p0)

    def psi22(self, f):
        """Aligned PhenomD phase Psi_22(f) and dPsi_22/df (both w.r.t. Mf)."""
        f = np.asarray(f, dtype=np.float64)
        pi_, dpi_ = self._psi_ins_raw(f)
        pm_, dpm_ = self._psi_int_raw(f)
        pm_ = pm_ + self.C1_int + self.C2_int * f
        dpm_ = dpm_ + self.C2_int
        pr_, dpr_ = self._psi_mr_raw(f)
        pr_ = pr_ + self.C1_mr + self.C2_mr * f
        dpr_ = dpr_ + self.C2_mr
        psi = np.where(f < F_PHI_INS, pi_, np.where(f < self.f_mr, pm_, pr_))
        dpsi = np.where(f < F_PHI_INS, dpi_, np.where(f < self.f_mr, dpm_, dpr_))
        psi = psi - self.p_shift - self.t_shift * (f - self.f_ref)
        dpsi = dpsi - self.t_shift
        return psi, dpsi

    # -------------------------------------------------------- higher modes
    def _map(self, l, m, f, for_amp):
        """O3 piecewise-linear map f -> f_22 and its (a_r, b_r) per point."""
        f = np.asarray(f, dtype=np.float64)
        f_i22 = F_AMP_INS if for_amp else F_PHI_INS
        f_i = 0.5 * m * f_i22
        f_r = self.f_rd[(l, m)]
        a_i, b_i = 2.0 / m, 0.0
        a_m = (self.fRD - f_i22) / (f_r - f_i)
        b_m = f_i22 - a_m * f_i
        if for_amp:
            a_r, b_r = 1.0, self.fRD - f_r
        else:
            a_r = self.fDM / self.f_damp[(l, m)]
            b_r = self.fRD - a_r * f_r
        a = np.where(f < f_i, a_i, np.where(f < f_r, a_m, a_r))
        b = np.where(f < f_i, b_i, np.where(f < f_r, b_m, b_r))
        return a, b, (f_i, f_r, (a_i, b_i), (a_m, b_m), (a_r, b_r))

    def beta_lm(self, l, m, f):
        """Leading-PN frequency-domain mode amplitude pi sqrt(2 eta/3) V^-7/2 |H_lm(V)|, V=(2 pi f/m)^(1/3)."""
        f = np.asarray(f, dtype=np.float64)
        V = (2.0 * PI * f / m) ** (1.0 / 3.0)
        c = self.table[f"hm.{l}{m}.amp"]
        eta, d = self.eta, self.delta
        H = {(2, 2): c + 0.0 * V,
             (2, 1): c * d * V,
             (3, 3): c * d * V,
             (3, 2): c * (1.0 - 3.0 * eta) * V ** 2,
             (4, 4): c * (1.0 - 3.0 * eta) * V ** 2,
             (4, 3): c * d * (1.0 - 2.0 * eta) * V ** 3}[(l, m)]
        return PI * math.sqrt(2.0 * eta / 3.0) * V ** -3.5 * np.abs(H)

    def amp_lm(self, l, m, f):
        """A_lm(f) = A_22(f22) beta_lm(f)/beta_22(f22), f22 = amplitude map (O3)."""
        f = np.asarray(f, dtype=np.float64)
        a, b, _ = self._map(l, m, f, True)
        f22 = a * f + b
        return self.amp22(f22) * self.beta_lm(l, m, f) / self.beta_lm(2, 2, f22)

    def psi_lm(self, l, m, f):
        """Psi_lm(f) (so phi_lm = -Psi_lm) and dPsi_lm/df = Psi_22'(f22) (O3)."""
        f = np.asarray(f, dtype=np.float64)
        a, b, (f_i, f_r, (a_i, b_i), (a_m, b_m), (a_r, b_r)) = self._map(l, m, f, False)
        f22 = a * f + b
        p22, dp22 = self.psi22(f22)
        p_at_i = float(self.psi22(np.float64(a_i * f_i + b_i))[0])
        p_at_r = float(self.psi22(np.float64(a_m * f_r + b_m))[0])
        c_i = 0.0
        c_m = c_i + p_at_i * (1.0 / a_i - 1.0 / a_m)
        c_r = c_m + p_at_r * (1.0 / a_m - 1.0 / a_r)
        c = np.where(f < f_i, c_i, np.where(f < f_r, c_m, c_r))
        psi = p22 / a + c - self.table[f"hm.{l}{m}.dphi"]
        return psi, dp22

    def t_of_f(self, l, m, f_hz, t_coal):
        """eq. 6: t_lm(f) = t_coal - (1/2pi) dphi_lm/df, in seconds."""
        _, dpsi = self.psi_lm(l, m, np.asarray(f_hz) * self.M_s)
        return t_coal + self.M_s * dpsi / (2.0 * PI)
