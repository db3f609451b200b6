"""Mutation check of the integrator / wall pins (tests/test_oracle_pins_integrator.py) and of the R28 pins
(tests/test_oracle_pins_coincident.py): applies, one at a time, the one-token
mutations of oracle/sph_oracle.c that the pins' docstrings name to a copy of the repo under /tmp and checks that the named
test FAILS on the mutant.  Not collected by pytest (takes ~2 min); run by hand:  python tests/oracle_mutations.py [name ...]
It calls only oracle/ and tests/ (no CUDA path)."""
import os, shutil, subprocess, sys
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__))); TMP = "/tmp/sph_oracle_mutations"
MUTS = [
 ("a7 drift 0.5", "            for (int d = 0; d < 3; ++d) o->r[3 * i + d] += 0.5 * dt * o->v[3 * i + d];", "            for (int d = 0; d < 3; ++d) o->r[3 * i + d] += dt * o->v[3 * i + d];", "test_I1"),
 ("a9 drift 0.5", "                o->r[3 * i + d] += 0.5 * dt * o->v[3 * i + d];", "                o->r[3 * i + d] += dt * o->v[3 * i + d];", "test_I1"),
 ("a7 rho 0.5", "o->rho[i] += 0.5 * dt * o->drho_saved[i];", "o->rho[i] += dt * o->drho_saved[i];", "test_I2"),
 ("a11 rho 0.5", "o->rho[i] += 0.5 * dt * o->drho_dt[i]; o->drho_saved[i] = o->drho_dt[i];", "o->rho[i] += dt * o->drho_dt[i]; o->drho_saved[i] = o->drho_dt[i];", "test_I2"),
 ("saved handover", "o->drho_saved[i] = o->drho_dt[i];", "", "test_I2"),
 ("sweepB factor 2", "o->drho_dt[i] = hydro ? 2.0 * rho_i * sr : 0.0;", "o->drho_dt[i] = hydro ? rho_i * sr : 0.0;", "test_I2"),
 ("reinit wall loop", "            const double *rj = &o->rw[3 * o->fw_idx[q]];\n            double d0 = ri[0] - rj[0], d1 = ri[1] - rj[1], d2 = ri[2] - rj[2];\n            s += orc_Wd(&o->p, sqrt(d0 * d0 + d1 * d1 + d2 * d2), h);", "", "test_I3"),
 ("reinit W(0)", "        double s = orc_Wd(&o->p, 0.0, h);\n        const double *ri = &o->r_frz[3 * i];", "        double s = 0.0;\n        const double *ri = &o->r_frz[3 * i];", "test_I3"),
 ("wall UR 2", "double UR = -UL + 2.0 * uw;", "double UR = -UL + uw;", "test_I4"),
 ("wall Us-UL", "sr += Vw * (Us - UL) * ne * dW;", "sr += Vw * (Us - Ub) * ne * dW;", "test_I4"),
 ("wall pR sign", "                double pR = p_i - rho_i * (p->g[0] * riw[0] + p->g[1] * riw[1] + p->g[2] * riw[2]);\n                double rhoR", "                double pR = p_i + rho_i * (p->g[0] * riw[0] + p->g[1] * riw[1] + p->g[2] * riw[2]);\n                double rhoR", "test_I4"),
 ("riemann c0", "*Ustar = Ub + (pL - pR) / (c0 * rs);", "*Ustar = Ub + (pL - pR) / (rs);", "test_I4"),
 ("uw sign", "double uw = -(nw[0] * vw[0] + nw[1] * vw[1] + nw[2] * vw[2]);", "double uw = (nw[0] * vw[0] + nw[1] * vw[1] + nw[2] * vw[2]);", "test_I4"),
 ("momentum 2", "if (do_p) ap[d] += -(2.0 / m_i) * V_i * V_j * ps * e[d] * dW;", "if (do_p) ap[d] += -(1.0 / m_i) * V_i * V_j * ps * e[d] * dW;", "test_I5"),
 ("Eq13 sign", "double vstar = vbar - (Us - Ub) * e[d];", "double vstar = vbar + (Us - Ub) * e[d];", "test_I5"),
 ("ps Pbar", "*pstar = Pb + rhoL * rhoR * beta * du / rs;", "*pstar = rhoL * rhoR * beta * du / rs;", "test_I5"),
 ("R28 e_ij 0/0", "static double orc_inv_r(double r) { return r > 0.0 ? 1.0 / r : 0.0; }", "static double orc_inv_r(double r) { return 1.0 / r; }", "test_C1"),
 ("R28 F(0) = 0", "    return -5.0 * a / (h * h);\n}", "    return 0.0 * a / (h * h);\n}", "test_C1"),
 ("R28 F(0) const", "    return -5.0 * a / (h * h);\n}", "    return -5.0 * a / h;\n}", "test_C1"),
]
extra = sys.argv[1:]
src = open(os.path.join(ROOT,'oracle/sph_oracle.c')).read()
res=[]
for name, old, new, test in MUTS:
    if extra and not any(e in name for e in extra): continue
    assert src.count(old) == 1, (name, src.count(old))
    shutil.rmtree(TMP, ignore_errors=True)
    os.makedirs(TMP)
    for d in ('oracle','tests','paper_2512_09904_b200'):
        shutil.copytree(os.path.join(ROOT,d), os.path.join(TMP,d), ignore=shutil.ignore_patterns('*.so','__pycache__','csrc'))
    open(os.path.join(TMP,'oracle/sph_oracle.c'),'w').write(src.replace(old,new))
    tfile = 'tests/test_oracle_pins_coincident.py' if test.startswith('test_C') else 'tests/test_oracle_pins_integrator.py'
    r = subprocess.run([sys.executable,'-m','pytest','-x','-q',tfile,'-k',test,'-p','no:cacheprovider'], cwd=TMP, capture_output=True, text=True)
    failed = r.returncode != 0
    print(f"{name:20s} -> {test}: {'FAILS (good)' if failed else 'PASSES (bad!)'}"); sys.stdout.flush()
    res.append(failed)
print(all(res))
