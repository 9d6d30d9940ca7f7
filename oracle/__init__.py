"""CPU oracle for the non-RNS CKKS/BGV hot path of arxiv/paper_2607_05920 (LibFHE).

TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct Python (arbitrary-precision ints,
NumPy uint64 for its own NTT).  Only `tests/`, `__graft_entry__.smoke()` and bench.py's
`cpu_baseline` / `--impl reference` legs may import anything from this package; the product
package `paper_2607_05920_b200` never does, and this package never imports the product.
The two share no code: primes, roots, tables, CRT method and rounding code are written twice.

Modules
-------
ring     negacyclic product pm(a, b, M): the definition (Eq. 5-6) by
         schoolbook, and the oracle's own NTT route (Eq. 7-9, Eq. 1) for large N.
ntt      the oracle's own prime search / roots / forward+inverse negacyclic NTT (Eq. 8-9).
scheme   parameters, he_mult, relinearize (CKKS and BGV), rescale.
harness  keygen, symmetric encryption, decryption, CKKS encode/decode.
limbs    Python-int <-> uint32 limb array packing used by the tests (Eq. 22).

Pin status (see tests/test_oracle_pins.py and DESIGN.md section 4):
  ring.pm_schoolbook / ring.pm_ntt / scheme.polymul / scheme.he_mult : pinned
      (hand brute force N=4, monomials, closed form a=b=Q-1, Kronecker substitution through one
       big-int multiply, ring laws, schoolbook-vs-NTT, NTT vs direct Eq. 8 evaluation).
  scheme.rescale, scheme.relinearize_ckks, scheme.relinearize_bgv, scheme.modswitch_bgv : PARITY UNPINNED by the
      paper (it prints no formula and no worked value for them); they follow the readings in
      DESIGN.md section 3.  Those readings are pinned by hand-worked values (tests/golden/relin_hand.txt: round half up
      at the tie, centred r, centred k, the 19 -> 13 switch) and held by invariants R1-R5 (rounding interval, decryption
      identities, CKKS 2^-20 bound, BGV exactness mod t before and after a level drop, degenerate keys).
"""
