// fg_plan.hpp — host planner: graph -> UV-divergent subgraphs -> forests -> (F,G') terms -> element
// geometries -> Dirac coefficient tables -> numerator record stream; Deg/Z density tables.
// Pure host code (no CUDA).  PAPER.md = /root/reference/PAPER.md (arXiv:1909.08015).
#pragma once
#include <array>
#include <cstdint>
#include <string>
#include <vector>

#include "fg_tables.h"

namespace fg {

struct Graph {                       // one open electron path, n photons, external photon at v_x
  int n = 0, nv = 0, x = 0;
  std::vector<int> partner;          // partner[v]: other end of v's photon; -1 for v_x
  std::vector<std::array<int, 2>> ph;   // photons (a < b) sorted by a; line id of photon k is 2n + k
};

struct Sub { int a, b, type; bool chain; };   // vertex interval [a,b]; type 0 self-energy, 1 vertexlike

struct Tok { int kind; int id; };   // kind 0: photon chord end (id = own photon), 1: external index, 2: slot (id)
struct Slot { int e; int se; int xiq; };   // own electron line whose eta-row / A / A^q it uses; index into se_kids or -1

struct HGeom {
  int sub = 0; std::vector<int> kids;           // kid sub indices (ascending a)
  int ne = 0, l = 0; bool has_x = false;
  std::vector<int> own_e, own_ph;               // global line ids
  std::vector<int> eta, xiq;                    // per own electron line
  std::vector<Tok> toks; std::vector<Slot> slots;   // string order (outgoing end first)
  std::vector<int> se_kids, vc_kids;            // sub indices
};

struct HRecord {
  int nf, k, dst, flags; float cabs[2];
  uint8_t fidx[FG_MAXF], vidx[FG_KMAX];
  std::vector<double> coef;                     // tables (see FgRecHdr), padded to an even count
};

struct HNum {
  int geom, op, ncomp, nse;
  std::vector<HRecord> recs;
  std::vector<int> nodes;
  long n_coefs = 0, n_nonzero = 0;
  double exec_flops = 0, algo_flops = 0;
};

struct HNode { int num; std::vector<int> se_kid, vc_kid; };

struct HTerm { std::vector<int> members, ops; int gprime; int sign; int top; std::vector<int> geoms; };

struct PlanOpts {
  double C[4] = {0.9, 0.03, 0.01, 0.06};        // Calc 2
  double D = 0.75;
  int merge = 0;
  std::vector<double> deg_override;
  double rel_tol = 1e-12, abs_tol = 0.0, err_factor = 0.0;
  bool structure_only = false;                  // stop after the combinatorics and the density tables
};

struct HostPlan {
  Graph g; PlanOpts opts;
  int M = 0, merge_var = -1;
  std::vector<std::vector<int>> var_lines;
  std::vector<Sub> subs;                         // subs[0] = G
  std::vector<std::vector<int>> forests;
  std::vector<HTerm> terms;
  std::vector<HGeom> geoms;
  std::vector<HNum> nums;                        // sorted by (interval length of geom, geom)
  std::vector<HNode> nodes;
  std::vector<int> geom_order;                   // evaluation order of geometries (children first)
  std::vector<double> deg, Z1, Z3; double lnZfull[4];
  // flattened
  std::vector<FgGeomDev> d_geoms; std::vector<FgNumDev> d_nums; std::vector<FgNodeDev> d_nodes;
  std::vector<FgTermDev> d_terms; std::vector<int32_t> d_geom_num_begin; std::vector<unsigned char> d_chunks; std::vector<uint32_t> d_chunk_used;
  std::vector<int32_t> d_geom_voff; int vtot = 0, vmax = 1;
  int raw_slots = 0, scratch_slots = 0;
  long n_records = 0, n_coefs = 0, n_nonzero = 0;
  double algo_flops = 0, exec_flops = 0, plan_seconds = 0;
};

// returns FG_OK or an FG_E_* code; msg receives the detail
int graph_from_edges(const int32_t* edges /* n_edges x (u,v,kind) */, int n_edges, int ext_vertex, Graph& g, std::string& msg);
int build_plan(const Graph& g, const PlanOpts& opts, HostPlan& P, std::string& msg);
// coefficient table (over the subsets of `gaps`) of one matching of the element ([a,b] with the given children shrunk);
// returns the number of slots or an FG_E_* code
int dirac_table(const Graph& g, int a, int b, const std::vector<std::array<int, 2>>& kid_iv, int op, int comp,
                const std::vector<std::array<int, 2>>& pairs, int qslot, std::vector<double>& table, std::vector<int>& gaps, std::string& msg);

}  // namespace fg
