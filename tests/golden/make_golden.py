"""Writes tests/golden/two_level_closed_form.json — a worked example whose every number follows from a closed form,
not from any implementation (neither oracle/ nor the CUDA path is imported here).

System: 2 electrons in 4 spinors (o = 2 occupied {0,1}, v = 2 virtual {2,3}), diagonal Fock (eps_o, eps_o, eps_v, eps_v),
the only non-zero antisymmetrised integrals are <23||01> = K and its Hermitian / antisymmetric partners.  The reference
|01> couples to |23> only, so FCI is a 2 x 2 problem (CCSD is exact for two electrons):

    E_corr = Delta - S,  Delta = eps_v - eps_o,  S = sqrt(Delta^2 + |K|^2),  t2[23,01] = E_corr / conj(K),  t1 = 0
    excitation energies (= eigenvalues of the Jacobian A): S (four singly excited determinants), 2 S (|23>)

and for the one-body operator X = d (a+_2 a_0 + a+_0 a_2) the sum-over-states response function (Eq. 23-24,
PAPER.md:273-288; sign convention of DESIGN.md reading 9) is  <<X;X>>_z = -d^2 [ 1/(S - z) + 1/(S + z) ].
"""
import json
import math
import os

eps_o, eps_v, K, d = -1.0, 0.5, 0.3 + 0.4j, 0.7
Delta = eps_v - eps_o
S = math.sqrt(Delta * Delta + abs(K) ** 2)
E_corr = Delta - S
t2 = E_corr / K.conjugate()
zs = [0.0, 0.0773, 0.0773 + 0.0045j, 1.5 + 0.0045j]
out = {
    "citation": "closed form of the 2x2 FCI problem; response: Eq. 23-24 PAPER.md:273-288, Eq. 19-21 PAPER.md:163-187",
    "eps_o": eps_o, "eps_v": eps_v, "K": [K.real, K.imag], "d": d,
    "S": S, "E_corr": E_corr, "t2_23_01": [t2.real, t2.imag],
    "jacobian_eigenvalues": [S, S, S, S, 2 * S],
    "response": [{"z": [complex(z).real, complex(z).imag],
                  "XX": [(-d * d * (1 / (S - z) + 1 / (S + z))).real, (-d * d * (1 / (S - z) + 1 / (S + z))).imag]}
                 for z in zs],
}
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "two_level_closed_form.json"), "w") as fh:
    json.dump(out, fh, indent=1)
print(json.dumps(out, indent=1))
