"""B200-native hot path of arxiv/paper_2606_30985 (Heisenberg-picture PEPO Trotter update,
BP sweeps, Bethe evaluation).  See DESIGN.md; the C ABI is in include/pepo.h."""
