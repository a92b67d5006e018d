#!/usr/bin/env python
"""Mutation check of the oracle pins (test infrastructure; `python tests/mutation_check.py [word ...]`).

Applies one plausible mistake at a time to a COPY of the repository (under the system temp
directory), rebuilds the oracle there, runs the CPU suite (`-m "not gpu"`) and prints which tests
turn red.  A mistake that leaves the suite green is a hole in the pins.  The table this printed for
the committed pins is in DESIGN.md ("Pins of the oracle").  Do not run it beside another OpenMP job:
two oversubscribed OpenMP runs spin in each other's barriers.
"""
import os, shutil, subprocess, sys, tempfile
SRC=os.path.dirname(os.path.dirname(os.path.abspath(__file__))); DST=os.path.join(tempfile.gettempdir(), "grmhd_mutation_check")
if os.path.exists(DST): shutil.rmtree(DST)
shutil.copytree(SRC, DST, ignore=shutil.ignore_patterns(".git","gpurun_out","_work","*.ncu-rep","__pycache__"))
cpp=os.path.join(DST,"oracle/grmhd_ref.cpp")
orig=open(cpp).read()
M=[
 ("maxspeed over padded range", "      for (int k = 0; k < nz; k++)\n        for (int j = 0; j < ny; j++)\n          for (int i = 0; i < nx; i++) {\n            const size_t c = idx(i, j, k);\n            const Metric M = cell_metric(c);\n            double gu[3][3];",
                                "      for (int k = -1; k < nz + 1; k++)\n        for (int j = -1; j < ny + 1; j++)\n          for (int i = -1; i < nx + 1; i++) {\n            const size_t c = idx(i, j, k);\n            const Metric M = cell_metric(c);\n            double gu[3][3];"),
 ("dt: max over directions", "    double dtm = INFINITY;\n    for (int d = 0; d < 3; d++) dtm = std::min(dtm, dx[d] / maxspeed[d]);", "    double dtm = 0;\n    for (int d = 0; d < 3; d++) dtm = std::max(dtm, dx[d] / maxspeed[d]);"),
 ("dt: speed of wrong shift component", "lam[0] = M.alpha * (vd * (1.0 - a2) - root) / den - M.beta[d];\n  lam[1] = M.alpha * (vd * (1.0 - a2) + root) / den - M.beta[d];", "lam[0] = M.alpha * (vd * (1.0 - a2) - root) / den - M.beta[(d + 1) % 3];\n  lam[1] = M.alpha * (vd * (1.0 - a2) + root) / den - M.beta[(d + 1) % 3];"),
 ("step_until: no clipping", "    if (dt > t_end - h->t) dt = t_end - h->t;\n", ""),
 ("RK2: weights 0.25/0.75", "y[q] = 0.5 * Y0[r][q] + 0.5 * (y[q] + h * k2[r][q]);", "y[q] = 0.25 * Y0[r][q] + 0.75 * (y[q] + h * k2[r][q]);"),
 ("RK3: 0.75/0.25 swapped", "y[q] = 0.75 * Y0[r][q] + 0.25 * (y[q] + h * k2[r][q]);", "y[q] = 0.25 * Y0[r][q] + 0.75 * (y[q] + h * k2[r][q]);"),
 ("RK3: 1/3,2/3 swapped", "y[q] = (1.0 / 3.0) * Y0[r][q] + (2.0 / 3.0) * (y[q] + h * k3[r][q]);", "y[q] = (2.0 / 3.0) * Y0[r][q] + (1.0 / 3.0) * (y[q] + h * k3[r][q]);"),
 ("RK4: missing factor 2 on k3", "(k1[r][q] + 2.0 * k2[r][q] + 2.0 * k3[r][q] + k4[r][q])", "(k1[r][q] + 2.0 * k2[r][q] + k3[r][q] + k4[r][q]) * (6.0 / 5.0)"),
 ("RK4: third stage half step", "for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], h, k3[r], Y(r));", "for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], 0.5 * h, k3[r], Y(r));"),
 ("A_i ghost: copy instead of linear extrapolation", "                  2.0 * q[idx(J[0], J[1], J[2])] - q[idx(K2[0], K2[1], K2[2])];", "                  q[idx(J[0], J[1], J[2])];"),
 ("face floors: no velocity cap", "  if (v2 > v2max) {\n    const double f = std::sqrt(v2max / v2);\n    for (int i = 0; i < 3; i++) P[1 + i] *= f;\n  }", ""),
 ("face floors: cap in the flat norm", "    for (int j = 0; j < 3; j++) v2 += M.g[i][j] * P[1 + i] * P[1 + j];\n  const double v2max", "    for (int j = 0; j < 3; j++) v2 += (i == j) * P[1 + i] * P[1 + j];\n  const double v2max"),
 ("B~0: sqrt(gamma) dropped", "h->B0[d][c] = 0.5 * (h->sqrtg_cell(cm) * Bin[cm] + h->sqrtg_cell(c) * Bin[c]);", "h->B0[d][c] = 0.5 * (Bin[cm] + Bin[c]);"),
 ("B~0: sqrt(gamma) of the wrong cell", "h->B0[d][c] = 0.5 * (h->sqrtg_cell(cm) * Bin[cm] + h->sqrtg_cell(c) * Bin[c]);", "h->B0[d][c] = 0.5 * (h->sqrtg_cell(c) * Bin[cm] + h->sqrtg_cell(c) * Bin[c]);"),
 ("flatten: offset 0.7", "const double f = 10.0 * (dp1 / dp2 - 0.75);", "const double f = 10.0 * (dp1 / dp2 - 0.7);"),
 ("flatten: slope 5", "const double f = 10.0 * (dp1 / dp2 - 0.75);", "const double f = 5.0 * (dp1 / dp2 - 0.75);"),
 ("flatten: threshold 0.5", "std::fabs(dp1) > 0.33 * std::min(p[3], p[1])", "std::fabs(dp1) > 0.5 * std::min(p[3], p[1])"),
 ("flatten: velocity test flipped", "&& vm1 > vp1) {", "&& vm1 < vp1) {"),
 ("c2p1d: t^2/x as printed", "0.5 * (t * t / (x * x) + s * iw2)", "0.5 * (t * t / x + s * iw2)"),
 ("audit3: eq 41d without 1/Gamma", "eps = (z / (rho * W * W) - 1.0) / Gamma;", "eps = (z / (rho * W * W) - 1.0);"),
 ("audit3: eq 40b with +B^2/2 (1 - v^2)", "const double f2 = tau + D - 0.5 * B2 * (1.0 + v2) + BS2 / (2.0 * z2) - z + p;", "const double f2 = tau + D - 0.5 * B2 * (1.0 - v2) + BS2 / (2.0 * z2) - z + p;"),
 ("audit3: W cap rescales by f^2", "    for (int i = 0; i < 3; i++) v[i] *= f;\n    bits |= 8;", "    for (int i = 0; i < 3; i++) v[i] *= f * f;\n    bits |= 8;"),
 ("equivalent (no test can tell: rho and v are kept, so the recomputed D = rho W is the D that came in): pressure fix also resets D", "    if (bits & 8) U5[0] = U[0];  // the pressure fix alone leaves D untouched", "    U5[0] = U[0];"),
 ("audit3: undensitise in the step forgotten", "for (int r = 0; r < 5; r++) Uin[r] = U[r][c] / sg;  // undensitise, eq. (17)", "for (int r = 0; r < 5; r++) Uin[r] = U[r][c];"),
 ("audit3: get_cons returns the densitised variables", "tmp[c] = r < 5 ? h->U[r][c] / h->sqrtg_cell(c) : h->Bc[r - 5][c];", "tmp[c] = r < 5 ? h->U[r][c] : h->Bc[r - 5][c];"),
 ("audit2: face metric by the 2-point mean", "m[f] = (-met[f][c0] + 9.0 * met[f][c1] + 9.0 * met[f][c2] - met[f][c3]) / 16.0;", "m[f] = 0.5 * (met[f][c1] + met[f][c2]);"),
 ("audit2: metric derivative 2nd order", "return (8.0 * (p1 - m1) - (p2 - m2)) / (12.0 * dx[a]);", "return (p1 - m1) / (2.0 * dx[a]);"),
 ("audit2: flux-CT E_z with the wrong neighbour", "            const double Ez = 0.25 * (-FxBy[idx(i, j - 1, k)] - FxBy[c] +\n                                      FyBx[idx(i - 1, j, k)] + FyBx[c]);", "            const double Ez = 0.25 * (-FxBy[idx(i - 1, j, k)] - FxBy[c] +\n                                      FyBx[idx(i, j - 1, k)] + FyBx[c]);"),
 ("audit2: flux-CT E_y sign", "            kA[1][c] = -Ey;", "            kA[1][c] = Ey;"),
 ("audit2: S_tau K term without the factor 2 on beta K", "t0 += T0i[i] * (2.0 * bK - dalpha[i]);", "t0 += T0i[i] * (bK - dalpha[i]);"),
 ("audit2: B_c from the lower face only", "Bc[1][c] = 0.5 * (Bf[1][c] + Bf[1][idx(i, j + 1, k)]) / sg;", "Bc[1][c] = Bf[1][c] / sg;"),
 ("audit2: Lorenz damping without alpha", "kPsi[c] = -div - xi * vertex(i, j, k).alpha * Psi[c];", "kPsi[c] = -div - xi * Psi[c];"),
 ("audit2: UCT bracket dissipation sign", "  return (ap * vL * BL + am * vR * BR - ap * am * (BR - BL)) / (ap + am);", "  return (ap * vL * BL + am * vR * BR + ap * am * (BR - BL)) / (ap + am);"),
 ("audit: PPM interface coefficient 1/8", "qp = 0.5 * (q[2] + q[3]) - (dm_p - dm_0) / 6.0;  // q_{i+1/2}", "qp = 0.5 * (q[2] + q[3]) - (dm_p - dm_0) / 8.0;  // q_{i+1/2}"),
 ("audit: PPM MC slope limit 1x instead of 2x", "std::min(2.0 * std::fabs(dp), 2.0 * std::fabs(dm))", "std::min(1.0 * std::fabs(dp), 1.0 * std::fabs(dm))"),
 ("audit: PPM monotonisation overshoot fix on the wrong side", "if (D * m > D * D / 6.0) qm = 3.0 * q0 - 2.0 * qp;", "if (D * m > D * D / 6.0) qp = 3.0 * q0 - 2.0 * qm;"),
 ("audit: minmod takes the larger slope", "  const double m = std::min(std::fabs(a), std::fabs(b));\n  return a > 0.0 ? m : -m;", "  const double m = std::max(std::fabs(a), std::fabs(b));\n  return a > 0.0 ? m : -m;"),
 ("audit: eq 18 magnetic pressure b^2 instead of b^2/2", "  const double ptot = P[4] + 0.5 * s.b2;\n  F[0]", "  const double ptot = P[4] + 1.0 * s.b2;\n  F[0]"),
 ("audit: eq 18 induction flux sign", "F[5 + k] = B[k] * vt[d] / M.alpha - B[d] * vt[k] / M.alpha;", "F[5 + k] = B[k] * vt[d] / M.alpha + B[d] * vt[k] / M.alpha;"),
 ("audit: eq 18 tau flux without the alpha b^0 B^d/W term", "F[4] = U[4] * vt[d] / M.alpha + ptot * v[d] - s.ab0 * B[d] / s.W;", "F[4] = U[4] * vt[d] / M.alpha + ptot * v[d];"),
 ("audit: eq 22 tau without the (alpha b^0)^2 term", "U[4] = (s.rhoh + s.b2) * W2 - (P[4] + 0.5 * s.b2) - sq(s.ab0) - U[0];", "U[4] = (s.rhoh + s.b2) * W2 - (P[4] + 0.5 * s.b2) - U[0];"),
 ("audit: eq 13 b^2 without the (alpha b^0)^2 term", "s.b2 = (s.B2 + sq(s.ab0)) / sq(s.W);", "s.b2 = (s.B2) / sq(s.W);"),
 ("audit: speeds with v_A^2 = b^2/rho h", "const double va2 = s.b2 / (s.rhoh + s.b2);", "const double va2 = s.b2 / (s.rhoh);"),
 ("ghost fill: mirror instead of copy", "          src = (kind == 0) ? 0 : g + 1;", "          src = (kind == 0) ? -g - 1 : g + 1;"),
 ("ghost fill: upper side copies the wrong layer", "          src = (kind == 0) ? hi[a] : g - 1;", "          src = (kind == 0) ? hi[a] - 1 : g - 1;"),
 ("ghost fill: corners left out", "      lo[a] = glo; hi[a] = ghi;\n    }\n  }", "    }\n  }"),
 ("mask: i and k swapped", "h->mask[h->idx(i, j, k)] = mask[((size_t)(k + G) * sy + (j + G)) * sx + (i + G)];", "h->mask[h->idx(i, j, k)] = mask[((size_t)(std::min(i, h->nz - 1) + G) * sy + (j + G)) * sx + (std::min(k, h->nx - 1) + G)];"),
 ("mask: shifted by one cell in x", "h->mask[h->idx(i, j, k)] = mask[((size_t)(k + G) * sy + (j + G)) * sx + (i + G)];", "h->mask[h->idx(i, j, k)] = mask[((size_t)(k + G) * sy + (j + G)) * sx + (i + G - 1)];"),
 ("mask: ignored by con2prim", "const int bits = con2prim(Uin, B, M, o, have_mask && mask[c], P5, U5, &it,", "const int bits = con2prim(Uin, B, M, o, false, P5, U5, &it,"),
 ("LxF: sign of the dissipation term", "Fhat[r] = 0.5 * (GR + GL - cw * (UR[r] - UL[r]));", "Fhat[r] = 0.5 * (GR + GL + cw * (UR[r] - UL[r]));"),
 ("LxF: c_wave = min", "const double cw = std::max(cmax, cmin);", "const double cw = std::min(cmax, cmin);"),
 ("LxF: c_wave = c_max alone", "const double cw = std::max(cmax, cmin);", "const double cw = cmax;"),
 ("LxF: missing 1/2 on the dissipation", "Fhat[r] = 0.5 * (GR + GL - cw * (UR[r] - UL[r]));", "Fhat[r] = 0.5 * (GR + GL) - cw * (UR[r] - UL[r]);"),
 ("HLLE: cmax/cmin swapped on the fluxes", "Fhat[r] = (cmin * GR + cmax * GL - cmax * cmin * (UR[r] - UL[r])) / (cmax + cmin);", "Fhat[r] = (cmax * GR + cmin * GL - cmax * cmin * (UR[r] - UL[r])) / (cmax + cmin);"),
]
res={}
only=sys.argv[1:] 
for name,a,b in M:
    if only and not any(o in name for o in only): continue
    if orig.count(a)!=1:
        res[name]="PATTERN NOT FOUND x%d"%orig.count(a); print(name,res[name],flush=True); continue
    open(cpp,"w").write(orig.replace(a,b))
    so=os.path.join(DST,"oracle/libgrmhd_ref.so")
    if os.path.exists(so): os.remove(so)
    p=subprocess.run([sys.executable,"-m","pytest","tests","-q","-m","not gpu","-p","no:cacheprovider","--tb=no","-k","not multirank and not abi"],cwd=DST,capture_output=True,text=True)
    failed=[l.split(" ")[1] for l in p.stdout.splitlines() if l.startswith("FAILED")]
    res[name]=failed; print(name,"->",failed,flush=True)
open(cpp,"w").write(orig)
holes=[k for k,v in res.items() if not v and not k.startswith("equivalent")]
print("holes:", holes)
sys.exit(1 if holes else 0)
